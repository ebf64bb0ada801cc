// pilot_pass_mma.cu — the pass kernel with the tensor-core contraction (pilot_math_mode MMA), in a translation unit of
// its own because its CTA shape differs: 4 warps at 72 registers, 7 CTAs = 28 warps per SM. Once the contraction is on
// the tensor cores the gather is bound by load latency and by the L1 data path (85 % busy), not by issue slots, and
// warps hide that better than registers of prefetched taps; measured on config 4 (B200, ms per step): 16 warps per SM at
// 128 registers with 6 rounds of 16-byte taps in flight 11.27; 32 warps at 64 registers with 2 rounds in flight 10.29;
// 32-byte loads (LDG.256, half the rounds), 28 warps at 72 registers, 1 round in flight 9.60 (FFMA2 path: 11.89).
// Shares no code with oracle/.
#ifndef PILOT_MMA_THREADS
#define PILOT_MMA_THREADS 128
#define PILOT_MMA_MIN_BLOCKS 6
#endif
#ifndef PILOT_MMA_PIPE
#define PILOT_MMA_PIPE 0
#endif
#define PILOT_THREADS PILOT_MMA_THREADS
#define PILOT_MIN_BLOCKS PILOT_MMA_MIN_BLOCKS
#include "pilot_pass.cuh"

namespace {

typedef void (*pass_fn)(const PassArgs);

template <class T>
pass_fn pick_mma(int g) {
  switch (g) {
#ifndef PILOT_FAST_BUILD
    case 2: return photo_pass_kernel<T, 2, false, true>;
#endif
    case 4: return photo_pass_kernel<T, 4, false, true>;
    case 8: return photo_pass_kernel<T, 8, false, true>;
#ifndef PILOT_FAST_BUILD
    case 16: return photo_pass_kernel<T, 16, false, true>;
#endif
  }
  return nullptr;
}

}  // namespace

int pilot_internal::mma_pass_launch(pilot_dtype dtype, int lanes_per_unit, const PassArgs& A, void* stream) {
  pass_fn fn = dtype == PILOT_BF16 ? pick_mma<BF16Tag>(lanes_per_unit) : (dtype == PILOT_F16 ? pick_mma<F16Tag>(lanes_per_unit) : nullptr);
  if (!fn) return (int)cudaErrorInvalidValue;
  const size_t smem = gather_smem_for(lanes_per_unit, true);
  if (smem > 48 * 1024 - 2 * 1024 &&
      cudaFuncSetAttribute(reinterpret_cast<const void*>(fn), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return (int)cudaErrorInvalidValue;
  fn<<<dim3((unsigned)A.n_hyp, (unsigned)A.n_chunks), kThreads, smem, static_cast<cudaStream_t>(stream)>>>(A);
  return (int)cudaGetLastError();
}
