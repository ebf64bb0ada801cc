// pilot_pdl.cuh - programmatic dependent launch, shared by every kernel the library enqueues back to back on the caller's
// stream (pass kernel -> finalize_kernel -> next pass, init_state -> level kernels, seed -> ... -> top-k -> ... -> arg-min).
// Shares no code with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace pilot_internal {

// Every CTA signals at its start that the NEXT kernel of the stream may be scheduled, and waits at its start for the PREVIOUS
// one to have completed (griddepcontrol.wait also makes its memory visible), so the next kernel's CTAs are resident and
// waiting when the last CTAs of this one finish: the launch latency between two dependent launches (22 per step of config 4,
// 13 per frame of the paper's schedule) leaves the critical path. A predecessor that never signals (any kernel of the
// caller's) releases its dependents when it completes, and a successor launched without the attribute waits for the whole
// grid: the caller's stream order is untouched. Kernels launched with launch_pdl MUST begin with pdl_prologue().
__device__ __forceinline__ void pdl_prologue() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}
template <class Fn, class... Args>
inline cudaError_t launch_pdl(Fn fn, dim3 grid, unsigned threads, size_t smem, cudaStream_t st, const Args&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = dim3(threads, 1, 1); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, fn, args...);
}

}  // namespace pilot_internal
