// pilot_probe.cu — the build's own gather micro-benchmark: random, vec_bytes-aligned reads of
// vec_bytes (one bilinear tap of C channels: 64 B for C=32 bf16, 128 B for C=64 bf16; 256/512 B for a whole
// 2x2 footprint) from a buffer that is either L2-resident or much larger than L2. It gives the denominators the
// photo kernel's gather is compared with: the L2->SM random-gather peak and the HBM random-gather peak (which is
// below the streaming-copy peak of MEASURED_PEAKS.json). Same access shapes as the kernels: 16-byte ld.global.nc per
// lane (FFMA2 gather) and, for vectors of 64 bytes and more, 32-byte loads (LDG.256, the tensor-core gather); the
// vec_bytes/16 or /32 lanes of a group read one contiguous vector. The result is the better of the two: the LSU costs
// per load instruction up to 32 bytes per lane, so the wider load sets the ceiling (measured: 14.4 vs 16.8 TB/s from
// an L2-resident buffer).
#include "../../include/pilot_refine.h"

#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__device__ __forceinline__ uint32_t mix(uint32_t x) {          // counter-based hash (lowbias32)
  x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
  return x;
}

// WB = bytes per lane per load: 16 (LDG.128) or 32 (LDG.256)
template <int WB> __device__ __forceinline__ uint4 probe_load(const char* p);
template <> __device__ __forceinline__ uint4 probe_load<16>(const char* p) { return __ldg(reinterpret_cast<const uint4*>(p)); }
template <> __device__ __forceinline__ uint4 probe_load<32>(const char* p) {
  uint4 a, b;
  asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(p));
  return make_uint4(a.x ^ b.x, a.y ^ b.y, a.z ^ b.z, a.w ^ b.w);
}

template <int UNROLL, int WB>
__global__ void __launch_bounds__(256) gather_probe_kernel(const char* __restrict__ buf, uint32_t n_vec, int lanes_per_vec,
                                                           uint32_t vecs_per_thread_group, uint32_t seed, uint4* sink) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t group = tid / lanes_per_vec, sub = tid % lanes_per_vec;
  uint4 acc = make_uint4(0, 0, 0, 0);
  for (uint32_t i = 0; i < vecs_per_thread_group; i += UNROLL) {
    uint4 v[UNROLL];
#pragma unroll
    for (int u = 0; u < UNROLL; ++u) {
      uint32_t k = mix((group * vecs_per_thread_group + i + u) ^ seed) % n_vec;
      v[u] = probe_load<WB>(buf + ((size_t)k * lanes_per_vec + sub) * WB);
    }
#pragma unroll
    for (int u = 0; u < UNROLL; ++u) { acc.x ^= v[u].x; acc.y ^= v[u].y; acc.z ^= v[u].z; acc.w ^= v[u].w; }
  }
  if (acc.x == 0x12345678u && acc.y == 0x9abcdef0u) sink[0] = acc;   // never true in practice: keeps the loads alive
}


// ------------------------------------------------------------------ unit-shaped gather (round 2)
//
// The access shape of the tensor-core gather, without its arithmetic: a warp takes rounds of 8 random "units"; row-group
// g (4 lanes) reads the unit's 2 x 2 taps (two x-adjacent pixels on each of two map rows) and its reference row, each lane
// TB = px_bytes / 4 bytes of every vector (LDG.256 at 128-byte pixels). Variant 1 stages the same bytes through shared
// memory instead: lanes 0-7 issue the unit's three bulk copies (cp.async.bulk, 2 x 2 px_bytes + px_bytes, completion on an
// mbarrier per ring stage, kStages rounds in flight) and the row-groups read them back with LDS.128 - the "feature tiles
// staged via TMA or shared memory" variant of north_star, measured here so that the choice between the two is a number.

struct W8 { unsigned w[8]; };
template <int TB> __device__ __forceinline__ unsigned unit_load(const char* p);
template <> __device__ __forceinline__ unsigned unit_load<32>(const char* p) {
  W8 t;
  asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(t.w[0]), "=r"(t.w[1]), "=r"(t.w[2]), "=r"(t.w[3]), "=r"(t.w[4]), "=r"(t.w[5]), "=r"(t.w[6]), "=r"(t.w[7]) : "l"(p));
  return t.w[0] ^ t.w[1] ^ t.w[2] ^ t.w[3] ^ t.w[4] ^ t.w[5] ^ t.w[6] ^ t.w[7];
}
template <> __device__ __forceinline__ unsigned unit_load<16>(const char* p) {
  const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
  return v.x ^ v.y ^ v.z ^ v.w;
}

template <int TB>
__global__ void __launch_bounds__(128) unit_gather_ldg_kernel(const char* __restrict__ buf, uint32_t n_px, uint32_t row_px, int rounds,
                                                              uint32_t seed, unsigned* sink) {
  constexpr int PX = 4 * TB;
  const int lane = threadIdx.x & 31, g = lane >> 2, q = lane & 3;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  unsigned acc = 0;
  for (int r = 0; r < rounds; ++r) {
    const uint32_t u = (warp * (uint32_t)rounds + (uint32_t)r) * 8u + (uint32_t)g;
    const uint32_t px = mix(u ^ seed) % (n_px - row_px - 2u), rf = mix((u * 3u + 1u) ^ seed) % n_px;
    const char* p = buf + (size_t)px * PX + q * TB;
    const unsigned a0 = unit_load<TB>(p), a1 = unit_load<TB>(p + PX);
    const unsigned a2 = unit_load<TB>(p + (size_t)row_px * PX), a3 = unit_load<TB>(p + (size_t)row_px * PX + PX);
    const unsigned a4 = unit_load<TB>(buf + (size_t)rf * PX + q * TB);
    acc ^= a0 ^ a1 ^ a2 ^ a3 ^ a4;
  }
  if (acc == 0x12345678u) sink[0] = acc;       // never true in practice: keeps the loads alive
}

__device__ __forceinline__ void mbar_init(unsigned bar, int n) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(n)); }
__device__ __forceinline__ void mbar_expect(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile("{\n.reg .pred p;\nPILOT_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra PILOT_DONE;\nbra PILOT_WAIT;\nPILOT_DONE:\n}"
               ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_copy(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
  asm volatile("cp.async.bulk.shared::cta.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

constexpr int kStages = 3;
template <int TB> __host__ __device__ constexpr int staged_unit_bytes() { return 5 * 4 * TB + 16; }   // + 16: the 8 units of a round fall in distinct banks
template <int TB> __host__ __device__ constexpr int staged_warp_bytes() { return kStages * 8 * staged_unit_bytes<TB>() + 64; }

template <int TB>
__global__ void __launch_bounds__(128) unit_gather_staged_kernel(const char* __restrict__ buf, uint32_t n_px, uint32_t row_px, int rounds,
                                                                 uint32_t seed, unsigned* sink) {
  constexpr int PX = 4 * TB, UB = staged_unit_bytes<TB>();
  extern __shared__ __align__(128) char probe_smem[];
  const int lane = threadIdx.x & 31, g = lane >> 2, q = lane & 3, wib = threadIdx.x >> 5;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  char* ring = probe_smem + (size_t)wib * staged_warp_bytes<TB>();
  const unsigned ring_s = (unsigned)__cvta_generic_to_shared(ring);
  const unsigned bars = ring_s + kStages * 8 * UB;
  if (lane == 0)
    for (int s = 0; s < kStages; ++s) mbar_init(bars + 8 * s, 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncwarp();
  auto issue = [&](int r) {
    const int s = r % kStages;
    const unsigned bar = bars + 8 * s, dst0 = ring_s + s * 8 * UB;
    if (lane == 0) mbar_expect(bar, 8 * 5 * PX);
    __syncwarp();
    if (lane < 8) {
      const uint32_t u = (warp * (uint32_t)rounds + (uint32_t)r) * 8u + (uint32_t)lane;
      const uint32_t px = mix(u ^ seed) % (n_px - row_px - 2u), rf = mix((u * 3u + 1u) ^ seed) % n_px;
      const unsigned d = dst0 + lane * UB;
      bulk_copy(d, buf + (size_t)px * PX, 2 * PX, bar);
      bulk_copy(d + 2 * PX, buf + (size_t)(px + row_px) * PX, 2 * PX, bar);
      bulk_copy(d + 4 * PX, buf + (size_t)rf * PX, PX, bar);
    }
  };
  for (int r = 0; r < kStages - 1 && r < rounds; ++r) issue(r);
  unsigned acc = 0;
  for (int r = 0; r < rounds; ++r) {
    if (r + kStages - 1 < rounds) issue(r + kStages - 1);
    const int s = r % kStages;
    mbar_wait(bars + 8 * s, (unsigned)(r / kStages) & 1u);
    const char* p = ring + s * 8 * UB + g * UB + q * TB;
#pragma unroll
    for (int i = 0; i < 5; ++i) {
#pragma unroll
      for (int h = 0; h < TB / 16; ++h) {
        const uint4 v = *reinterpret_cast<const uint4*>(p + i * PX + h * 16);
        acc ^= v.x ^ v.y ^ v.z ^ v.w;
      }
    }
    __syncwarp();                     // every lane has read stage s before issue(r + kStages) refills it
  }
  if (acc == 0x12345678u) sink[0] = acc;
}

}  // namespace

extern "C" {

int pilot_refine_probe_gather(int device, size_t buffer_bytes, int vec_bytes, int launches, double* gbps_out) {
  if (!gbps_out || launches < 1 || vec_bytes < 16 || vec_bytes > 512 || (vec_bytes & (vec_bytes - 1)) ||
      buffer_bytes < (size_t)vec_bytes * 1024)
    return PILOT_ERR_ARG;
  int prev = 0;
  cudaGetDevice(&prev);
  if (cudaSetDevice(device) != cudaSuccess) return PILOT_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaSetDevice(prev); return PILOT_ERR_CUDA; }
  const size_t n_vec = buffer_bytes / vec_bytes;
  void *buf = nullptr, *sink = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  bool ok = n_vec <= 0xffffffffull && cudaMalloc(&buf, n_vec * vec_bytes) == cudaSuccess && cudaMalloc(&sink, 16) == cudaSuccess &&
            cudaMemset(buf, 1, n_vec * vec_bytes) == cudaSuccess && cudaEventCreate(&e0) == cudaSuccess &&
            cudaEventCreate(&e1) == cudaSuccess;
  double best = 0.0;
  if (ok) {
    const int ctas = prop.multiProcessorCount * 8;                 // 8 resident CTAs of 256 threads per SM
    const uint32_t per_group = 256;                                // vectors per lane group per launch
    for (int wb = 16; wb <= (vec_bytes >= 64 ? 32 : 16) && ok; wb *= 2) {
      const int lanes = vec_bytes / wb;
      const double bytes = (double)ctas * 256 / lanes * per_group * vec_bytes;
      for (int it = 0; it < launches + 2 && ok; ++it) {            // 2 warm-up launches (also fill L2 when it fits)
        cudaEventRecord(e0);
        const uint32_t seed = 0x9e3779b9u * (uint32_t)(it + 1);
        if (wb == 16)
          gather_probe_kernel<8, 16><<<ctas, 256>>>(static_cast<const char*>(buf), (uint32_t)n_vec, lanes, per_group, seed,
                                                    static_cast<uint4*>(sink));
        else
          gather_probe_kernel<8, 32><<<ctas, 256>>>(static_cast<const char*>(buf), (uint32_t)n_vec, lanes, per_group, seed,
                                                    static_cast<uint4*>(sink));
        cudaEventRecord(e1);
        ok = cudaEventSynchronize(e1) == cudaSuccess && cudaGetLastError() == cudaSuccess;
        float ms = 0.f;
        if (ok && it >= 2 && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess && ms > 0.f) {
          double g = bytes / (ms * 1e-3) / 1e9;
          if (g > best) best = g;
        }
      }
    }
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (buf) cudaFree(buf);
  if (sink) cudaFree(sink);
  cudaSetDevice(prev);
  *gbps_out = best;
  return ok ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_probe_unit_gather(int device, size_t buffer_bytes, int px_bytes, int variant, int launches, double* gbps_out) {
  if (!gbps_out || launches < 1 || (px_bytes != 64 && px_bytes != 128) || variant < 0 || variant > 1 ||
      buffer_bytes < (size_t)px_bytes * 65536 || buffer_bytes / px_bytes > 0xffffffffull)
    return PILOT_ERR_ARG;
  int prev = 0;
  cudaGetDevice(&prev);
  if (cudaSetDevice(device) != cudaSuccess) return PILOT_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaSetDevice(prev); return PILOT_ERR_CUDA; }
  const uint32_t n_px = (uint32_t)(buffer_bytes / px_bytes), row_px = 1920;
  void *buf = nullptr, *sink = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  bool ok = cudaMalloc(&buf, (size_t)n_px * px_bytes) == cudaSuccess && cudaMalloc(&sink, 16) == cudaSuccess &&
            cudaMemset(buf, 1, (size_t)n_px * px_bytes) == cudaSuccess && cudaEventCreate(&e0) == cudaSuccess &&
            cudaEventCreate(&e1) == cudaSuccess;
  double best = 0.0;
  const int rounds = 512;
  // resident CTAs of 4 warps per SM: as many as the kernel it stands for can hold (variant 0), or as shared memory allows
  const int smem = variant == 1 ? 4 * (px_bytes == 128 ? staged_warp_bytes<32>() : staged_warp_bytes<16>()) : 0;
  if (ok && variant == 1) {
    ok = (px_bytes == 128 ? cudaFuncSetAttribute(unit_gather_staged_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)
                          : cudaFuncSetAttribute(unit_gather_staged_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) == cudaSuccess;
  }
  const int occ_list[3] = {6, 8, 12};
  for (int oi = 0; oi < 3 && ok; ++oi) {
    int occ = occ_list[oi];
    if (variant == 1) { const int fit = (int)((prop.sharedMemPerMultiprocessor - 4096) / (size_t)(smem + 1024)); if (oi > 0) break; occ = fit < 1 ? 1 : fit; }
    const int ctas = prop.multiProcessorCount * occ;
    const double tap_bytes = (double)ctas * 4 * rounds * 8 * 4 * px_bytes;
    for (int it = 0; it < launches + 2 && ok; ++it) {
      const uint32_t seed = 0x9e3779b9u * (uint32_t)(it + 1);
      cudaEventRecord(e0);
      if (variant == 0) {
        if (px_bytes == 128) unit_gather_ldg_kernel<32><<<ctas, 128>>>(static_cast<const char*>(buf), n_px, row_px, rounds, seed, static_cast<unsigned*>(sink));
        else unit_gather_ldg_kernel<16><<<ctas, 128>>>(static_cast<const char*>(buf), n_px, row_px, rounds, seed, static_cast<unsigned*>(sink));
      } else {
        if (px_bytes == 128) unit_gather_staged_kernel<32><<<ctas, 128, smem>>>(static_cast<const char*>(buf), n_px, row_px, rounds, seed, static_cast<unsigned*>(sink));
        else unit_gather_staged_kernel<16><<<ctas, 128, smem>>>(static_cast<const char*>(buf), n_px, row_px, rounds, seed, static_cast<unsigned*>(sink));
      }
      cudaEventRecord(e1);
      ok = cudaEventSynchronize(e1) == cudaSuccess && cudaGetLastError() == cudaSuccess;
      float ms = 0.f;
      if (ok && it >= 2 && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess && ms > 0.f) {
        const double gb = tap_bytes / (ms * 1e-3) / 1e9;
        if (gb > best) best = gb;
      }
    }
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (buf) cudaFree(buf);
  if (sink) cudaFree(sink);
  cudaSetDevice(prev);
  *gbps_out = best;
  return ok ? PILOT_OK : PILOT_ERR_CUDA;
}

}  // extern "C"
