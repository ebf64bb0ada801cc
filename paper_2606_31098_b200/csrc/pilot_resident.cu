// pilot_resident.cu — the cluster-resident LM kernel for small problems (latency-bound regime: the paper's own
// frame shape of 10^2-10^3 hypotheses x 500 anchors; BASELINE configs 0, 1, 3).
//
// One launch per pyramid LEVEL instead of one per EVAL pass: a thread-block cluster of S CTAs owns one hypothesis
// for all of that level's LM iterations (hypotheses are independent, so clusters never wait on each other).
// Per iteration: every CTA gathers its slice of the anchors (same photo_accumulate as the pass kernel), reduces it
// to 32 floats in shared memory and SENDS them to EVERY CTA of the cluster (asynchronous DSMEM stores that complete on the
// receiver's mbarrier: an all-gather of S x 128 bytes); every CTA's warp 0 waits for the S slices, sums them in the same
// fixed order (deterministic), adds the priors, takes the accept/reject decision, solves the damped 6x6 system and
// retracts (finalize_hypothesis, shared with the pass kernel) on ITS OWN replica of the optimiser state - the replicas stay
// bit-identical, so the new candidate pose is simply there, in every CTA's shared memory, without travelling (round 2,
// earlier: rank 0 alone finalised and sent the pose back, one more hand-off per iteration on the critical path). There is
// no cluster-wide barrier inside the loop: only the threads that need a hand-off wait for it.
// The heightfield ray-march of the range prior and the algebra of both priors (their terms of supp Eq.5-6) depend only
// on the candidate pose, so one warp of the rank-0 CTA evaluates them WHILE the other warps gather and its 28 numbers
// travel with rank 0's slice: they leave the critical path. The optimiser state lives in shared memory for the whole level; launches, grid ramps, the atomic
// ticket and the global partial sums of the pass kernel disappear.
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
  HypState st;                       // EVERY rank keeps a replica of the hypothesis' optimiser state and finalises it itself
  __align__(16) double pose[12];     // candidate pose Rc[9], Cc[3] of this iteration (written by this CTA's own finaliser)
  float posef[16];                   // right behind the pose: R, centre hi, centre lo as floats (pose_to_float)
  int go;                            // 1 = evaluate this pose, 0 = the level is finished
  float part[kWarps][kNacc];
  __align__(16) float slice[2][8][kNacc];   // by iteration parity: the slice totals of every rank, written by their owners (DSMEM)
  double tot[kNacc];                 // the cluster's sums, converted to double by the lane that added each
  PriorTerms prior[2];               // by iteration parity: what the priors add at the candidate pose (rank 0's prior warp sends it)
  PriorTerms stage_prior;            // rank 0: where its prior warp leaves the terms before warp 0 sends them
  unsigned long long bar_sums[2];    // mbarriers by iteration parity: S x 128 bytes (+ the prior terms) per use
};
constexpr unsigned kSliceBytes = kNacc * 4, kPriorBytes = (unsigned)sizeof(PriorTerms);
static_assert(sizeof(PriorTerms) % 8 == 0, "the prior terms travel as 8-byte messages");

// ---- cluster hand-off: asynchronous DSMEM stores that complete on the CONSUMER's mbarrier (st.async ...
// mbarrier::complete_tx::bytes): the data and its arrival are one message, so the producer needs no fence and only the
// threads that need the data wait. Every rank sends its slice total to EVERY rank (an all-gather of S x 128 bytes), and every
// rank's warp 0 sums the slices in the same fixed order and runs the same finalisation on its own replica of the state: the
// candidate pose never travels (measured, config 1 | config 3 | paper schedule, ms per step: two cluster.sync() per
// iteration 0.504 | 0.850 | 0.251; slices to rank 0 + the pose back by st.async 0.468 | 0.809 | 0.242 before the fp32
// projection, 0.458 | 0.781 | 0.240 after it; this all-gather: see profiles/r2_resident_config1.md). Barriers and slice
// buffers alternate with the iteration parity: a rank that runs ahead writes into the other buffer, and it cannot be two
// iterations ahead because its next iteration needs this rank's slice.
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned map_rank(unsigned addr, unsigned rank) {
  unsigned r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
// the local arrival of a phase: so many bytes of asynchronous stores are expected before it completes
__device__ __forceinline__ void mbar_arm(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "PILOT_WAIT:\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
      "@p bra PILOT_DONE;\n"
      "bra PILOT_WAIT;\n"
      "PILOT_DONE:\n"
      "}\n" ::"r"(smem_addr(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void st_async(unsigned dst, unsigned long long v, unsigned bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];" ::"r"(dst), "l"(v), "r"(bar) : "memory");
}
__device__ __forceinline__ void st_async(unsigned dst, unsigned v, unsigned bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];" ::"r"(dst), "r"(v), "r"(bar) : "memory");
}

// The candidate pose of the next evaluation from this CTA's replica of the state, into this CTA's shared memory (doubles,
// the float copy the fp32 projection reads, and the go flag). Call with one warp.
__device__ __forceinline__ void stage_pose(ResidentShared& sh, int lane, int level) {
  if (lane < 9) sh.pose[lane] = sh.st.Rc[lane];
  else if (lane < 12) sh.pose[lane] = sh.st.Cc[lane - 9];
  else if (lane >= 16) pose_to_float(sh.st.Rc, sh.st.Cc, lane - 16, sh.posef);
  if (lane == 12) sh.go = sh.st.level == level ? 1 : 0;
}

template <class T, int G, bool CEN, bool MMA>
__global__ void __launch_bounds__(kThreads, PILOT_MIN_BLOCKS) lm_resident_kernel(const __grid_constant__ PassArgs A) {
  pdl_prologue();
  cg::cluster_group cluster = cg::this_cluster();
  const unsigned S = cluster.num_blocks(), rank = cluster.block_rank();
  const int m = (int)(blockIdx.x / S);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  __shared__ ResidentShared sh;
  PILOT_DECLARE_ACC

  const bool range_on = range_enabled(A);
  const unsigned expect = S * kSliceBytes + (range_on ? kPriorBytes : 0u);
  if (threadIdx.x == 0) {
    mbar_init(&sh.bar_sums[0], 1u);
    mbar_init(&sh.bar_sums[1], 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  {
    const int* src = reinterpret_cast<const int*>(A.state + m);
    int* dst = reinterpret_cast<int*>(&sh.st);
    for (int i = threadIdx.x; i < (int)(sizeof(HypState) / 4); i += kThreads) dst[i] = src[i];
  }
  __syncthreads();
  if (warp == 0) stage_pose(sh, lane, A.level);
  cluster.sync();                                    // every CTA of the cluster runs and its barriers are initialised
  const bool prior_warp = range_on && rank == 0 && warp == kWarps - 1;
  // the gathering warps of the whole cluster share the anchors: worker w of n_workers (rank 0's last warp evaluates the
  // priors instead) - 32-anchor batches round-robin
  const int n_workers = (int)S * kWarps - (range_on ? 1 : 0);
  const int worker = (int)rank * kWarps + warp - ((range_on && rank > 0) ? 1 : 0);
  const int N = A.lv.N;

#ifdef PILOT_RESIDENT_PROFILE
  long long t_eval = 0, t_fin = 0, t_red = 0, t_all = clock64(), t0 = 0, n_it = 0;
#endif
  for (unsigned it = 0;; ++it) {
    const unsigned par = it & 1u, wait_parity = (it >> 1) & 1u;
    __syncthreads();                                 // this iteration's pose is in sh.pose (this CTA's warp 0 wrote it)
#ifdef PILOT_RESIDENT_PROFILE
    t0 = clock64();
#endif
    if (!*(volatile int*)&sh.go) break;
    if (threadIdx.x == 0) mbar_arm(&sh.bar_sums[par], expect);   // this CTA's arrival; the bytes may already be coming in

    acc_zero<MMA>(acc, sacc);
    if (prior_warp) {
      // the priors' terms at the candidate pose, computed WHILE the others gather, then sent to every rank
      prior_terms_store(A, sh.pose, sh.pose + 9, lane, &sh.stage_prior);
    } else {
      photo_accumulate<T, G, CEN, MMA>(A, sh.pose, sh.pose + 9, 0, N, worker, n_workers, acc, sacc, red);
    }
    const float wtot = acc_warp_total<MMA>(acc, sacc, lane);
#ifdef PILOT_RESIDENT_PROFILE
    t_eval += clock64() - t0; t0 = clock64();
#endif
    sh.part[warp][lane] = wtot;
    __syncthreads();
    if (warp != 0) continue;
    {
      float t = 0.f;
#pragma unroll
      for (int w = 0; w < kWarps; ++w) t += sh.part[w][lane];            // fixed order
      const unsigned dst0 = smem_addr(&sh.slice[par][rank][lane]), bar0 = smem_addr(&sh.bar_sums[par]);
      for (unsigned r = 0; r < S; ++r) st_async(map_rank(dst0, r), __float_as_uint(t), map_rank(bar0, r));
      if (range_on && rank == 0) {                   // rank 0 also sends the prior terms its last warp left in sh.stage_prior
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(&sh.stage_prior);
        const unsigned dstp = smem_addr(&sh.prior[par]);
        for (unsigned r = 0; r < S; ++r)
          for (unsigned i = (unsigned)lane; i < kPriorBytes / 8u; i += 32u) st_async(map_rank(dstp, r) + 8u * i, src[i], map_rank(bar0, r));
      }
    }
    mbar_wait(&sh.bar_sums[par], wait_parity);       // every rank's slice total (and the prior terms) of this iteration
#ifdef PILOT_RESIDENT_PROFILE
    t_red += clock64() - t0; t0 = clock64(); ++n_it;
#endif
    {
      float t = 0.f;
#pragma unroll
      for (unsigned r = 0; r < 8; ++r) t += r < S ? *(volatile float*)&sh.slice[par][r][lane] : 0.f;   // fixed order
      sh.tot[lane] = (double)t;
      __syncwarp();
      finalize_hypothesis(A, sh.st, m, sh.tot, lane, range_on ? &sh.prior[par] : nullptr);
      __syncwarp();
      stage_pose(sh, lane, A.level);
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
  cluster.sync();                                    // nobody's shared memory goes away while a peer may still write to it
  if (rank == 0) {                                   // the state goes back to the workspace for the next level
    const int* src = reinterpret_cast<const int*>(&sh.st);
    int* dst = reinterpret_cast<int*>(A.state + m);
    for (int i = threadIdx.x; i < (int)(sizeof(HypState) / 4); i += kThreads) dst[i] = src[i];
  }
}

typedef void (*resident_fn)(const PassArgs);

template <class T, bool CEN>
resident_fn pick_g(int g) {
  switch (g) {
    case 1: return lm_resident_kernel<T, 1, CEN, false>;
    case 2: return lm_resident_kernel<T, 2, CEN, false>;
    case 4: return lm_resident_kernel<T, 4, CEN, false>;
    case 8: return lm_resident_kernel<T, 8, CEN, false>;
    case 16: return lm_resident_kernel<T, 16, CEN, false>;
    case 32: return lm_resident_kernel<T, 32, CEN, false>;
  }
  return nullptr;
}

template <class T>
resident_fn pick_mma(int g) {
  switch (g) {
    case 2: return lm_resident_kernel<T, 2, false, true>;
    case 4: return lm_resident_kernel<T, 4, false, true>;
    case 8: return lm_resident_kernel<T, 8, false, true>;
    case 16: return lm_resident_kernel<T, 16, false, true>;
  }
  return nullptr;
}

template <bool CEN>
resident_fn pick_t(pilot_dtype d, int g) {
  switch (d) {
    case PILOT_F32: return pick_g<F32Tag, CEN>(g);
    case PILOT_F16: return pick_g<F16Tag, CEN>(g);
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
  if (smem > 40 * 1024 &&                            // dynamic + the kernel's ~5 KB of static shared memory must not exceed the default 48 KB
      cudaFuncSetAttribute(reinterpret_cast<const void*>(fn), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return (int)cudaErrorInvalidValue;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = static_cast<cudaStream_t>(stream);
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cluster;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see pdl_prologue (pilot_device.cuh)
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  return (int)cudaLaunchKernelEx(&cfg, fn, A);
}
