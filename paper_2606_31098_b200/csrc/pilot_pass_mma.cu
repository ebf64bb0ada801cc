// pilot_pass_mma.cu — the pass kernel with the tensor-core contraction (pilot_math_mode MMA), in a translation unit of
// its own because its CTA shape differs from the FFMA2 kernel's: 4 warps at 80 registers, 6 CTAs = 24 warps per SM (the
// finalisation is out of line, so the hot loop fits without spills). With one unit per row-group (pilot_device.cuh) the
// gather runs at the rate at which the L1 takes missed 128-byte lines (about 1.85 clocks per line per SM, the ceiling of
// pilot_refine_probe_unit_gather), and warps hide that better than registers of prefetched taps. Measured on config 4
// (B200, ms per step): 16 warps at 128 registers 8.76 (8.31 with the next round's taps prefetched), 20 warps at 96: 8.17,
// 24 at 80: 7.88, 28 at 72: 7.94, 32 at 64: 8.30; CTAs of 2 / 8 warps at the same occupancy 7.94 / 8.02; anchors per CTA
// 768 ... 3072: 7.83-7.87 (1536 kept). Round 1's layout (a unit split over two row-groups, 28 warps at 72 registers): 7.65
// with the empty batches skipped, 8.98 without. Later changes of round 2 (staged finalisation, fp32 projection, product-major
// Gram order: pilot_device.cuh) took the 7.88 of this sweep to 7.00 at the same shape; re-checked then: 72 / 64 registers
// 7.51 / 8.76, super-batch 64 / 128: 7.14 / 7.73, anchors per CTA 1024 ... 2304: 7.03-7.25. Shares no code with oracle/.
#ifndef PILOT_MMA_THREADS
#define PILOT_MMA_THREADS 128
#define PILOT_MMA_MIN_BLOCKS 6
#endif
#ifndef PILOT_MMA_PIPE
#define PILOT_MMA_PIPE 0
#endif
#ifndef PILOT_MMA_PROJ_ILP
#define PILOT_MMA_PROJ_ILP 1
#endif
#ifndef PILOT_MMA_SB
#define PILOT_MMA_SB 96             // anchors per super-batch of a warp: measured (B200, config 4 | config 2, ms) 32: 8.00 | 7.76,
                                    // 64: 7.77 | 7.50, 96: 7.75 | 7.41, 128: 8.50 | 7.62
#endif
#define PILOT_THREADS PILOT_MMA_THREADS
#define PILOT_MIN_BLOCKS PILOT_MMA_MIN_BLOCKS
#include "pilot_pass.cuh"

namespace {

typedef void (*pass_fn)(const PassArgs);

template <class T>
pass_fn pick_mma(int g) {
  switch (g) {
    case 2: return photo_pass_kernel<T, 2, false, true>;
    case 4: return photo_pass_kernel<T, 4, false, true>;
    case 8: return photo_pass_kernel<T, 8, false, true>;
    case 16: return photo_pass_kernel<T, 16, false, true>;
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
  return (int)launch_pdl(fn, dim3((unsigned)A.n_hyp, (unsigned)(A.n_chunks + A.prior_cta)), kThreads, smem,
                         static_cast<cudaStream_t>(stream), A);
}
