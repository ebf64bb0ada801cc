// pilot_resident.cu — the cluster-resident LM kernel for small problems (latency-bound regime: the paper's own
// frame shape of 10^2-10^3 hypotheses x 500 anchors; BASELINE configs 0, 1, 3).
//
// One launch per pyramid LEVEL instead of one per EVAL pass: a thread-block cluster of S CTAs owns one hypothesis
// for all of that level's LM iterations (hypotheses are independent, so clusters never wait on each other).
// Per iteration: every CTA gathers its slice of the anchors (same photo_accumulate as the pass kernel), reduces it
// to 32 floats in shared memory; after a cluster barrier the rank-0 CTA sums the S slices through distributed
// shared memory in a fixed order (deterministic), adds the priors, takes the accept/reject decision, solves the
// damped 6x6 system and retracts (finalize_hypothesis, shared with the pass kernel); a second cluster barrier
// publishes the new candidate pose, which the other CTAs read from rank 0's shared memory. The heightfield
// ray-march of the range prior and the algebra of both priors (their terms of supp Eq.5-6) depend only on the candidate
// pose, so one warp of the rank-0 CTA evaluates them WHILE the other warps gather: they leave the critical path. The optimiser state lives in shared memory for the
// whole level; launches, grid ramps, the atomic ticket and the global partial sums of the pass kernel disappear.
//
// Shares no code with oracle/.
#ifndef PILOT_MMA_SB
#define PILOT_MMA_SB 128            // anchors per super-batch of a warp (10 KB of shared memory per warp at 2 CTAs per SM)
#endif
#include "pilot_device.cuh"

#include <cooperative_groups.h>
#include <string.h>

namespace cg = cooperative_groups;

namespace {

struct ResidentShared {
  HypState st;                       // rank 0: the hypothesis' optimiser state for the whole level
  __align__(16) double pose[12];     // this CTA's copy of the candidate pose: Rc[9], Cc[3]
  float part[kWarps][kNacc];
  float cta_sum[kNacc];              // this CTA's slice total; rank 0 reads it through DSMEM
  double tot[kNacc];                 // the cluster's sums, converted to double by the lane that added each
  PriorTerms prior;                  // what the priors add at the candidate pose (the prior warp writes it during the gather)
  int go;
};

template <class T, int G, bool CEN, bool MMA>
__global__ void __launch_bounds__(kThreads, PILOT_MIN_BLOCKS) lm_resident_kernel(const __grid_constant__ PassArgs A) {
  cg::cluster_group cluster = cg::this_cluster();
  const unsigned S = cluster.num_blocks(), rank = cluster.block_rank();
  const int m = (int)(blockIdx.x / S);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  __shared__ ResidentShared sh;
  PILOT_DECLARE_ACC

  if (rank == 0) {
    const int* src = reinterpret_cast<const int*>(A.state + m);
    int* dst = reinterpret_cast<int*>(&sh.st);
    for (int i = threadIdx.x; i < (int)(sizeof(HypState) / 4); i += kThreads) dst[i] = src[i];
    __syncthreads();
    if (threadIdx.x == 0) sh.go = sh.st.level == A.level;
  }
  const ResidentShared* master = cluster.map_shared_rank(&sh, 0);
  const bool range_on = range_enabled(A);
  const bool prior_warp = range_on && rank == 0 && warp == kWarps - 1;
  // the gathering warps of the whole cluster share the anchors: worker w of n_workers (rank 0's last warp evaluates the
  // range prior instead) - contiguous equal ranges on the tensor-core path, 32-anchor batches round-robin on the FFMA2 path
  const int n_workers = (int)S * kWarps - (range_on ? 1 : 0);
  const int worker = (int)rank * kWarps + warp - ((range_on && rank > 0) ? 1 : 0);
  const int N = A.lv.N;

#ifdef PILOT_RESIDENT_PROFILE
  long long t_eval = 0, t_fin = 0, t_red = 0, t_all = clock64(), t0 = 0, n_it = 0;
#endif
  for (;;) {
    cluster.sync();                                  // rank 0's candidate pose and go flag are published
#ifdef PILOT_RESIDENT_PROFILE
    t0 = clock64();
#endif
    const int go = master->go;
    if (threadIdx.x < 12) sh.pose[threadIdx.x] = threadIdx.x < 9 ? master->st.Rc[threadIdx.x] : master->st.Cc[threadIdx.x - 9];
    __syncthreads();
    if (!go) break;

    acc_zero<MMA>(acc, sacc);
    if (prior_warp) {
      prior_terms_store(A, sh.pose, sh.pose + 9, lane, &sh.prior);
    } else {
      photo_accumulate<T, G, CEN, MMA>(A, sh.pose, sh.pose + 9, 0, N, worker, n_workers, acc, sacc, red);
    }
    const float wtot = acc_warp_total<MMA>(acc, sacc, lane);
#ifdef PILOT_RESIDENT_PROFILE
    t_eval += clock64() - t0; t0 = clock64();
#endif
    sh.part[warp][lane] = wtot;
    __syncthreads();
    if (warp == 0) {
      float t = 0.f;
#pragma unroll
      for (int w = 0; w < kWarps; ++w) t += sh.part[w][lane];            // fixed order
      sh.cta_sum[lane] = t;
    }
    cluster.sync();                                  // every slice total (and the prior) is in shared memory
#ifdef PILOT_RESIDENT_PROFILE
    t_red += clock64() - t0; t0 = clock64(); ++n_it;
#endif
    if (rank == 0 && warp == 0) {
      float v[8];
#pragma unroll
      for (unsigned r = 0; r < 8; ++r) v[r] = r < S ? cluster.map_shared_rank(&sh, r)->cta_sum[lane] : 0.f;   // loads in flight together
      float t = 0.f;
#pragma unroll
      for (unsigned r = 0; r < 8; ++r) t += v[r];                         // fixed order
      sh.tot[lane] = (double)t;
      __syncwarp();
      finalize_hypothesis(A, sh.st, m, sh.tot, lane, range_on ? &sh.prior : nullptr);
      __syncwarp();
      if (lane == 0) sh.go = sh.st.level == A.level;
#ifdef PILOT_RESIDENT_PROFILE
      t_fin += clock64() - t0;
#endif
    }
  }
#ifdef PILOT_RESIDENT_PROFILE
  if (rank == 0 && (threadIdx.x == 0 || threadIdx.x == kThreads - 1 || threadIdx.x == 32)) {
    float* o = A.partials + (size_t)m * 32 + (threadIdx.x == 0 ? 0 : (threadIdx.x == 32 ? 8 : 16));
    o[0] = (float)t_eval; o[1] = (float)t_red; o[2] = (float)t_fin; o[3] = (float)(clock64() - t_all); o[4] = (float)n_it;
  }
#endif
  if (rank == 0) {                                   // the state goes back to the workspace for the next level
    const int* src = reinterpret_cast<const int*>(&sh.st);
    int* dst = reinterpret_cast<int*>(A.state + m);
    for (int i = threadIdx.x; i < (int)(sizeof(HypState) / 4); i += kThreads) dst[i] = src[i];
  }
  cluster.sync();                                    // rank 0's shared memory outlives every remote read
}

typedef void (*resident_fn)(const PassArgs);

template <class T, bool CEN>
resident_fn pick_g(int g) {
  switch (g) {
#ifndef PILOT_FAST_BUILD
    case 1: return lm_resident_kernel<T, 1, CEN, false>;
#endif
#ifndef PILOT_FAST_BUILD
    case 2: return lm_resident_kernel<T, 2, CEN, false>;
#endif
    case 4: return lm_resident_kernel<T, 4, CEN, false>;
    case 8: return lm_resident_kernel<T, 8, CEN, false>;
#ifndef PILOT_FAST_BUILD
    case 16: return lm_resident_kernel<T, 16, CEN, false>;
#endif
#ifndef PILOT_FAST_BUILD
    case 32: return lm_resident_kernel<T, 32, CEN, false>;
#endif
  }
  return nullptr;
}

template <class T>
resident_fn pick_mma(int g) {
  switch (g) {
#ifndef PILOT_FAST_BUILD
    case 2: return lm_resident_kernel<T, 2, false, true>;
#endif
    case 4: return lm_resident_kernel<T, 4, false, true>;
    case 8: return lm_resident_kernel<T, 8, false, true>;
#ifndef PILOT_FAST_BUILD
    case 16: return lm_resident_kernel<T, 16, false, true>;
#endif
  }
  return nullptr;
}

template <bool CEN>
resident_fn pick_t(pilot_dtype d, int g) {
  switch (d) {
#ifndef PILOT_FAST_BUILD      /* tuning builds (-DPILOT_FAST_BUILD): bf16, 32 and 64 channels only */
    case PILOT_F32: return pick_g<F32Tag, CEN>(g);
    case PILOT_F16: return pick_g<F16Tag, CEN>(g);
#endif
    case PILOT_BF16: return pick_g<BF16Tag, CEN>(g);
  }
  return nullptr;
}

}  // namespace

int pilot_internal::resident_launch(pilot_dtype dtype, int lanes_per_unit, int grad_mode, bool mma, const PassArgs& A,
                                    int cluster, void* stream) {
  resident_fn fn = mma ? (dtype == PILOT_BF16 ? pick_mma<BF16Tag>(lanes_per_unit) : pick_mma<F16Tag>(lanes_per_unit))
                       : (grad_mode == PILOT_GRAD_CENTRAL_SAMPLED ? pick_t<true>(dtype, lanes_per_unit)
                                                                  : pick_t<false>(dtype, lanes_per_unit));
  if (!fn || cluster < 1 || cluster > 8 || (cluster & (cluster - 1))) return (int)cudaErrorInvalidValue;
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof cfg);
  cfg.gridDim = dim3((unsigned)A.n_hyp * (unsigned)cluster, 1, 1);
  cfg.blockDim = dim3(kThreads, 1, 1);
  const size_t smem = gather_smem_for(lanes_per_unit, mma);
  if (smem > 48 * 1024 - 3 * 1024 &&
      cudaFuncSetAttribute(reinterpret_cast<const void*>(fn), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return (int)cudaErrorInvalidValue;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = static_cast<cudaStream_t>(stream);
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cluster;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return (int)cudaLaunchKernelEx(&cfg, fn, A);
}
