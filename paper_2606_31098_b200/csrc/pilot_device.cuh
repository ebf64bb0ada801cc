// pilot_device.cuh — device code shared by the two launch strategies of the refinement (pilot_refine.cu: one
// launch per EVAL pass, many CTAs per hypothesis; pilot_resident.cu: one launch per pyramid level, a thread-block
// cluster owns a hypothesis for all of its LM iterations). Everything here is in an anonymous namespace: each
// translation unit gets its own copy. Shares no code with oracle/.
#pragma once
#include "../../include/pilot_refine.h"

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <math.h>

#include "pilot_pdl.cuh"
#include <stdint.h>
#include <type_traits>

namespace {

// Tuning knobs of the photo gather (compile time). Defaults = the combination measured fastest on B200 over
// configs 1-4 (round 1: registers/prefetch 1 12.47 | 0.727 ms, shared/prefetch 2 12.45 | 0.681 ms on config 4 |
// config 1; 3 CTAs per SM at 80 registers spills and gains 1.5 % on config 4 but loses 10 % on config 1).
#ifndef PILOT_PREFETCH
#define PILOT_PREFETCH 2        // units of a lane group whose taps are in flight ahead of the arithmetic (1 or 2)
#endif
#ifndef PILOT_SMEM_ACC
#define PILOT_SMEM_ACC 1        // 1: the 29 per-thread accumulators live in shared memory (a [32][256] fp32 array, one
                                // conflict-free column per thread) so that the registers they held carry prefetched taps
#endif
#ifndef PILOT_SMEM_RS
#define PILOT_SMEM_RS 1         // 1: the per-unit sum over a lane group's channel slices goes through a shared-memory
                                // transpose (3 STS.64 per round + 1.5 G LDS.128 + 6 (G-1) FADD per batch) instead of the
                                // shuffle reduce-scatter (6 (G-1) x (SHFL + 2 FSEL + FADD)); used for 2 <= G <= 8
#endif
#ifndef PILOT_MIN_BLOCKS
#define PILOT_MIN_BLOCKS 2      // resident CTAs per SM the kernels are compiled for (register cap 128 / 85)
#endif

#ifndef PILOT_THREADS
#define PILOT_THREADS 256
#endif
constexpr int kThreads = PILOT_THREADS;   // threads per CTA of the gather kernels
constexpr int kWarps = kThreads / 32;
constexpr int kNacc = 32;                // 21 H + 6 g + cost + n_valid, padded to 32 floats
constexpr int kMinChunk = kWarps * 32;   // one 32-unit batch per warp

// index of the upper-triangular entry (a<=b) in the packed 21-vector
__host__ __device__ constexpr int tri(int a, int b) { return a * 6 - a * (a - 1) / 2 + (b - a); }

}  // namespace

namespace pilot_internal {   // types that cross translation units (pilot_refine.cu <-> pilot_resident.cu)

// Per-hypothesis optimiser state, device resident (workspace).
struct HypState {
  double R[9], C[3];        // accepted pose: R_cw row-major, camera centre
  double Rc[9], Cc[3];      // candidate pose evaluated by the next pass
  double H[21], g[6];       // accepted total system (upper triangle), undamped
  double cost;              // accepted total cost (Eq.7)
  double lambda;
  int n_valid;
  unsigned flags;           // FEW_VALID / RANGE_SKIP of the accepted state
  unsigned status;          // sticky bits
  int level;                // pyramid level this hypothesis is in (n_levels = finished)
  int k;                    // solves consumed at this level
  int pending;              // 1 if (Rc, Cc) came from a solve (not the level's first evaluation)
  unsigned long long visible_evals;   // measurement: visible (anchor, hypothesis) units summed over every EVAL pass of the run
};

struct LevelArgs {
  const void* feat;         // [H][W][C]
  const float* conf;        // [H][W] or null
  const float4* points;     // [N] xyz + w_ref
  const void* ref;          // [N][C]
  float fx, fy, cx, cy;
  int W, H, C, N;
};

struct PassArgs {
  LevelArgs lv;
  pilot_refine_params prm;
  // priors
  float gw[3], gi[3], ray[3], range_meas;
  const float* dsm; int dsm_w, dsm_h; float dsm_ox, dsm_oy, dsm_gsd;
  // run
  int n_hyp, level, level_end, pass, iters, rec_base;
  int chunk, n_chunks;
  int defer;                // 1: the pass kernel only writes partial sums; finalize_kernel ends the iteration
  int prior_cta;            // 1 (only with defer): row 0 of the grid's y axis is one CTA per hypothesis that evaluates the priors'
                            // terms at the candidate pose WHILE the other rows gather; finalize_kernel adds them (struct PriorTerms)
  void* priors;             // [n_hyp] PriorTerms in the workspace
  // what the finalisation reads as doubles, converted once on the host (an F2F costs the single finalising lane ~18 cycles)
  struct { double lambda_init, lambda_up, lambda_down, lambda_min, lambda_max, w_gravity, gravity_scale, w_range, range_scale,
                  gw[3], gi[3]; } pd;
  HypState* state;
  float* partials;          // [n_hyp][n_chunks][kNacc]
  unsigned* counters;       // [n_hyp]
  pilot_refine_outputs out;
  // optional extra records (pilot_refine_set_iterate_outputs; NULL = off)
  float* iter_poses;        // [sum(iters)][n_hyp][12]: the accepted pose [R_wc | C] each recorded system was built at
  int* iter_accept;         // [sum(iters)][n_hyp]: 1 if the step solved from that record was accepted
};

// pilot_resident.cu: one launch of the cluster-resident LM kernel for the level described by A (A.lv, A.level,
// A.iters, A.rec_base): `cluster` CTAs per hypothesis. Returns a cudaError_t as int.
int resident_launch(pilot_dtype dtype, int lanes_per_unit, int grad_mode, bool mma, const PassArgs& A, int cluster, void* stream);

// pilot_pass_mma.cu: one launch of the pass kernel with the tensor-core contraction (grid = A.n_hyp x A.n_chunks).
int mma_pass_launch(pilot_dtype dtype, int lanes_per_unit, const PassArgs& A, void* stream);

}  // namespace pilot_internal
using namespace pilot_internal;

namespace {

// ------------------------------------------------------------------ element decoding

struct F32Tag { static constexpr int kVec = 4; };
struct BF16Tag { static constexpr int kVec = 8; };
struct F16Tag { static constexpr int kVec = 8; };

__device__ __forceinline__ uint4 ldg16(const void* p) {
  return __ldg(reinterpret_cast<const uint4*>(p));
}

// ------------------------------------------------------------------ fast double reciprocal / reciprocal sqrt
//
// A double-precision divide or sqrt is a ~30-instruction dependent sequence (measured on B200, one warp, dependent chain:
// 1/x 59 cycles, sqrt 78; a dependent DFMA 8). The per-hypothesis finalisation (one lane, the serial tail of every LM
// iteration), the ray-march and the projection of every anchor are chains of them. These start from the fp64 hardware
// seed (MUFU.RCP64H / MUFU.RSQ64H: 2^-22 relative, no fp32 round trip) and take ONE third-order step in double: relative
// error <= 2.6e-16 over 2^-100 .. 2^100, 40 / 50 cycles (round 1's fp32 seed + two Newton steps: 161 / 155).
// Arguments outside 2^-1007 .. 2^993 in magnitude (zero, subnormal, inf, NaN) take the exact division on a cold branch.
__device__ __forceinline__ bool fp64_mid_range(double d) {
  const unsigned hi = (unsigned)__double2hiint(d) & 0x7fffffffu;
  return hi - 0x01000000u < 0x7e000000u - 0x01000000u;
}
__device__ __forceinline__ double inv_sqrt_core(double s) {       // s > 0 in the middle range
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
  const double t = s * y;
  const double e = fma(-t, y, 1.0);                               // 1 - s y^2
  const double p = fma(0.375, e, 0.5), ye = y * e;
  return fma(ye, p, y);                                           // y (1 + e/2 + 3 e^2 / 8)
}
__device__ __forceinline__ double inv_sqrt(double s) {
  if (!fp64_mid_range(s) || s < 0.0) return 1.0 / sqrt(s);
  return inv_sqrt_core(s);
}
__device__ __forceinline__ double fast_rcp(double d) {
  if (!fp64_mid_range(d)) return 1.0 / d;
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
  const double e = fma(-d, y, 1.0);                               // 1 - d y
  const double p = fma(e, e, e);
  return fma(y, p, y);                                            // y (1 + e + e^2)
}

// rho, rho' for the prior terms, in double, without sqrt / divide
__device__ __forceinline__ void robust_d(int loss, double x, double scale, double& rho, double& drho) {
  rho = x; drho = 1.0;
  if (scale > 0.0) {
    const double s2 = scale * scale;
    if (loss == PILOT_LOSS_HUBER) {
      if (x > s2) { const double y = inv_sqrt(x); rho = 2.0 * scale * (x * y) - s2; drho = scale * y; }
    } else if (loss == PILOT_LOSS_CAUCHY) {
      const double q = x * fast_rcp(s2);
      rho = s2 * log1p(q);
      drho = fast_rcp(1.0 + q);
    }
  }
}

// ------------------------------------------------------------------ robust loss (Eq.2 / Eq.7)

template <typename T>
__device__ __forceinline__ void robust(int loss, T x, T scale, T& rho, T& drho) {
  rho = x; drho = T(1);
  if (scale > T(0)) {
    T s2 = scale * scale;
    if (loss == PILOT_LOSS_HUBER) {
      if (x > s2) { T sq = sqrt(x); rho = T(2) * scale * sq - s2; drho = scale / sq; }
    } else if (loss == PILOT_LOSS_CAUCHY) {
      T q = x / s2;
      rho = s2 * log1p(q);
      drho = T(1) / (T(1) + q);
    }
  }
}

// The same for the 16-bit feature path, whose tolerance (5e-3) leaves room for the hardware approximations: rsqrt / rcp /
// lg2 (MUFU, ~2^-22 relative) instead of the divide, sqrt and log1p sequences. log(1 + q) through lg2 loses RELATIVE
// accuracy for tiny q (6e-8 / q), but its ABSOLUTE error per unit is <= 6e-8 s^2, nothing against a cost of ~N s^2.
__device__ __forceinline__ void robust_fast(int loss, float x, float scale, float& rho, float& drho) {
  rho = x; drho = 1.f;
  if (scale > 0.f) {
    const float s2 = scale * scale;
    if (loss == PILOT_LOSS_HUBER) {
      if (x > s2) { const float y = rsqrtf(x); rho = 2.f * scale * (x * y) - s2; drho = scale * y; }
    } else if (loss == PILOT_LOSS_CAUCHY) {
      const float q1 = 1.f + x * __frcp_rn(s2);
      rho = s2 * 0.69314718056f * __log2f(q1);
      drho = __frcp_rn(q1);
    }
  }
}

}  // namespace

namespace {

// ------------------------------------------------------------------ gather of one unit by a lane group
//
// The G = C*sizeof/16 lanes of a group own one (anchor, hypothesis) unit: each lane loads 16 B of
// every bilinear tap (the four taps of a unit are 2 x 2 pixels x C channels = 4*C*s bytes, the
// algorithmic gather traffic) and of the reference feature, and returns its share of
//   p = { gx.gx, gx.gy, gy.gy, gx.r, gy.r, r.r }.
struct RawTaps { uint4 q00, q10, q01, q11, ref; };

template <int PX>   // PX = bytes per pixel = 16*G: the x+1 taps are an immediate offset away
__device__ __forceinline__ RawTaps load_taps(const char* feat, unsigned off, unsigned row_stride, const char* ref) {
  RawTaps t;
  const char* p = feat + off;
  const char* q = p + row_stride;
  t.q00 = ldg16(p);
  t.q10 = ldg16(p + PX);
  t.q01 = ldg16(q);
  t.q11 = ldg16(q + PX);
  t.ref = ldg16(ref);
  return t;
}

// Packed fp32x2 arithmetic (sm_100 FFMA2 / FADD2): two channels per instruction, half the issue slots.
__device__ __forceinline__ float2 sub2(float2 x, float2 y) { return __ffma2_rn(y, make_float2(-1.f, -1.f), x); }

template <class T> __device__ __forceinline__ void unpack2(const uint4& v, float2 (&o)[T::kVec / 2]);
template <> __device__ __forceinline__ void unpack2<F32Tag>(const uint4& v, float2 (&o)[2]) {
  o[0] = make_float2(__uint_as_float(v.x), __uint_as_float(v.y));
  o[1] = make_float2(__uint_as_float(v.z), __uint_as_float(v.w));
}
template <> __device__ __forceinline__ void unpack2<BF16Tag>(const uint4& v, float2 (&o)[4]) {
  // a 32-bit word holds channels (2i, 2i+1): low half << 16 and the masked high half are the two fp32 values
  o[0] = make_float2(__uint_as_float(v.x << 16), __uint_as_float(v.x & 0xffff0000u));
  o[1] = make_float2(__uint_as_float(v.y << 16), __uint_as_float(v.y & 0xffff0000u));
  o[2] = make_float2(__uint_as_float(v.z << 16), __uint_as_float(v.z & 0xffff0000u));
  o[3] = make_float2(__uint_as_float(v.w << 16), __uint_as_float(v.w & 0xffff0000u));
}
template <> __device__ __forceinline__ void unpack2<F16Tag>(const uint4& v, float2 (&o)[4]) {
  const __half2* h = reinterpret_cast<const __half2*>(&v);
#pragma unroll
  for (int i = 0; i < 4; ++i) o[i] = __half22float2(h[i]);
}

template <class T>
__device__ __forceinline__ void unit_partials(const RawTaps& t, float a, float b, float (&p)[6]) {
  constexpr int V2 = T::kVec / 2;
  float2 f00[V2], f10[V2], f01[V2], f11[V2], fr[V2];
  unpack2<T>(t.q00, f00); unpack2<T>(t.q10, f10); unpack2<T>(t.q01, f01); unpack2<T>(t.q11, f11);
  unpack2<T>(t.ref, fr);
  const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
  float2 acc[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) acc[i] = make_float2(0.f, 0.f);
#pragma unroll
  for (int i = 0; i < V2; ++i) {
    float2 d0 = sub2(f10[i], f00[i]);          // x-difference, top row
    float2 d1 = sub2(f11[i], f01[i]);          // x-difference, bottom row
    float2 top = __ffma2_rn(a2, d0, f00[i]);
    float2 bot = __ffma2_rn(a2, d1, f01[i]);
    float2 gy = sub2(bot, top);                // = (1-a)(f01-f00) + a(f11-f10): exact d/dv of the bilinear patch
    float2 f = __ffma2_rn(b2, gy, top);        // bilinear value
    float2 gx = __ffma2_rn(b2, sub2(d1, d0), d0);  // = (1-b)(f10-f00) + b(f11-f01): exact d/du
    float2 r = sub2(f, fr[i]);                 // Eq.(1)
    acc[0] = __ffma2_rn(gx, gx, acc[0]);
    acc[1] = __ffma2_rn(gx, gy, acc[1]);
    acc[2] = __ffma2_rn(gy, gy, acc[2]);
    acc[3] = __ffma2_rn(gx, r, acc[3]);
    acc[4] = __ffma2_rn(gy, r, acc[4]);
    acc[5] = __ffma2_rn(r, r, acc[5]);
  }
#pragma unroll
  for (int i = 0; i < 6; ++i) p[i] = acc[i].x + acc[i].y;
}

// GRAD_CENTRAL_SAMPLED (reading A7): gx, gy = bilinear sample (same a, b) of the central-difference
// maps Dx[y][x] = 0.5 (F[y][min(x+1,W-1)] - F[y][max(x-1,0)]), Dy likewise (replicate border), computed on the fly
// from the 4x4-minus-corners footprint. `nb` holds the byte offsets of the clamped outer taps relative to the
// top-left tap: x-1 | x+2 (pixels), y-1 | y+2 (rows). The value f uses the same 2x2 taps as the default mode.
struct OuterTaps { int xl, xr, yu, yd; };

template <class T, int PX>
__device__ __forceinline__ void unit_partials_central(const char* p00, unsigned row_stride, const OuterTaps& nb,
                                                      const char* ref, float a, float b, float (&p)[6]) {
  constexpr int V2 = T::kVec / 2;
  const char* p01 = p00 + row_stride;
  float2 f00[V2], f10[V2], f01[V2], f11[V2], t0[V2], t1[V2], t2[V2], t3[V2];
  unpack2<T>(ldg16(p00), f00); unpack2<T>(ldg16(p00 + PX), f10);
  unpack2<T>(ldg16(p01), f01); unpack2<T>(ldg16(p01 + PX), f11);
  const float2 a2 = make_float2(a, a), b2 = make_float2(b, b), h2 = make_float2(0.5f, 0.5f);
  float2 gx[V2], gy[V2], r[V2];
  // Dx at the four taps: 0.5 (right - left); right of x0 is x0+1, left of x0+1 is x0
  unpack2<T>(ldg16(p00 + nb.xl), t0); unpack2<T>(ldg16(p00 + nb.xr), t1);
  unpack2<T>(ldg16(p01 + nb.xl), t2); unpack2<T>(ldg16(p01 + nb.xr), t3);
#pragma unroll
  for (int i = 0; i < V2; ++i) {
    float2 dx00 = sub2(f10[i], t0[i]), dx10 = sub2(t1[i], f00[i]);
    float2 dx01 = sub2(f11[i], t2[i]), dx11 = sub2(t3[i], f01[i]);
    float2 top = __ffma2_rn(a2, sub2(dx10, dx00), dx00);
    float2 bot = __ffma2_rn(a2, sub2(dx11, dx01), dx01);
    gx[i] = __fmul2_rn(h2, __ffma2_rn(b2, sub2(bot, top), top));
  }
  // Dy: 0.5 (below - above); below of y0 is y0+1, above of y0+1 is y0
  unpack2<T>(ldg16(p00 + nb.yu), t0); unpack2<T>(ldg16(p00 + nb.yd), t1);
  unpack2<T>(ldg16(p00 + PX + nb.yu), t2); unpack2<T>(ldg16(p00 + PX + nb.yd), t3);
#pragma unroll
  for (int i = 0; i < V2; ++i) {
    float2 dy00 = sub2(f01[i], t0[i]), dy01 = sub2(t1[i], f00[i]);
    float2 dy10 = sub2(f11[i], t2[i]), dy11 = sub2(t3[i], f10[i]);
    float2 top = __ffma2_rn(a2, sub2(dy10, dy00), dy00);
    float2 bot = __ffma2_rn(a2, sub2(dy11, dy01), dy01);
    gy[i] = __fmul2_rn(h2, __ffma2_rn(b2, sub2(bot, top), top));
  }
  unpack2<T>(ldg16(ref), t0);
  float2 acc[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) acc[i] = make_float2(0.f, 0.f);
#pragma unroll
  for (int i = 0; i < V2; ++i) {
    float2 top = __ffma2_rn(a2, sub2(f10[i], f00[i]), f00[i]);
    float2 bot = __ffma2_rn(a2, sub2(f11[i], f01[i]), f01[i]);
    float2 f = __ffma2_rn(b2, sub2(bot, top), top);
    r[i] = sub2(f, t0[i]);
    acc[0] = __ffma2_rn(gx[i], gx[i], acc[0]);
    acc[1] = __ffma2_rn(gx[i], gy[i], acc[1]);
    acc[2] = __ffma2_rn(gy[i], gy[i], acc[2]);
    acc[3] = __ffma2_rn(gx[i], r[i], acc[3]);
    acc[4] = __ffma2_rn(gy[i], r[i], acc[4]);
    acc[5] = __ffma2_rn(r[i], r[i], acc[5]);
  }
#pragma unroll
  for (int i = 0; i < 6; ++i) p[i] = acc[i].x + acc[i].y;
}

// One step of a recursive-halving reduce-scatter across lane bit `bit`: lanes with the bit clear
// keep `lo`, lanes with it set keep `hi`; each receives the partner's copy of what it keeps.
template <int N>
__device__ __forceinline__ void halve(float (&lo)[N], const float (&hi)[N], int bit, bool upper) {
#pragma unroll
  for (int i = 0; i < N; ++i) {
    float send = upper ? lo[i] : hi[i];
    float keep = upper ? hi[i] : lo[i];
    lo[i] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
  }
}

template <int G> struct Log2 { static constexpr int v = 1 + Log2<G / 2>::v; };
template <> struct Log2<1> { static constexpr int v = 0; };

// Shared-memory transpose of the group reduction: row u of a warp's buffer holds, for unit u of the batch, the six
// partial sums of each of the G lanes ([G][6] floats). Row stride = 6 G rounded up to an odd multiple of 4 words, so
// that the 32 lanes' LDS.128 of their own rows are conflict-free.
template <int G> struct RedRows {
  static constexpr bool kOn = PILOT_SMEM_RS && G >= 2 && G <= 8;
  static constexpr int kStride = G == 2 ? 12 : (G == 4 ? 28 : (G == 8 ? 52 : 0));
  // The lane groups that store in the same half-warp phase would hit the same banks (G * kStride is a multiple of 32
  // words): every group's block of rows is shifted by kSkew more words than the previous one (a multiple of 4, so
  // rows stay 16-B aligned; cumulative, so rows never overlap).
  static constexpr int kSkew = G == 8 ? 16 : (G == 4 ? 4 : 0);
  static constexpr int kWarpFloats = kOn ? 32 * kStride + kSkew * (32 / G) : 0;
  __device__ static __forceinline__ int row(int u) { return u * kStride + kSkew * (u / G); }
};
// ------------------------------------------------------------------ tensor-core variant of the per-unit contraction
//
// For 16-bit features the C x 3 contraction of a unit (a3-a5) is a 4 x 4 Gram matrix E = D D^T of FIRST DIFFERENCES
//   e0 = f10 - f00,  e1 = f11 - f01,  e2 = f01 - f00,  e3 = ref - f01          (rows of D, C channels each)
// followed by three quadratic forms in the bilinear weights (gram_unit_scalars below):
//   gx = (1-b) e0 + b e1,   gy = -a e0 + a e1 + e2,   r = f - ref = a(1-b) e0 + ab e1 + (b-1) e2 - e3.
// The differences are taken in the storage type (packed HSUB2: exact whenever the two values are within a factor of two
// of each other - Sterbenz - which is every channel of a smooth map except at zero crossings; otherwise one rounding of
// 2^-9 (bf16) / 2^-12 (fp16) relative to the DIFFERENCE, not to the taps), their products are exact and accumulate in
// fp32 on the tensor cores (mma.sync.m16n8k16 = HMMA.16816.F32). Differencing first is what makes the Gram safe: a
// Gram of the raw taps would cancel by ~3e4.
//
// Fragment roles (round 2): ONE UNIT PER ROW-GROUP. Thread (g, q) of the fragment layout (g = lane / 4, q = lane % 4)
// loads, for the unit of row-group g, its quarter of the pixel (C/2 bytes: one 32-byte LDG.256 at C = 64) of ALL FIVE
// vectors - the four q-threads of a row-group read one whole pixel per instruction, 8 units = 8 lines per warp-wide load,
// and no vector is fetched twice (round 1 split a unit over two row-groups, which cost a second fetch of f01 and a
// 16-float hand-off per unit). It forms the four differences for its channels and issues, per 16-channel k-step,
//   A = {e0 | e2} (rows g | g+8) x B = e0, e1, e3, e2      and      A' = {e1 | e3} x B = e1, e3
// (B column g = the same thread's registers): the diagonal entries C[g][g], C[g+8][g] of the six accumulators are the
// ten distinct entries of E for unit g (two come twice), and they all land in ONE thread, (g, q = g / 2).
template <class T> struct MmaType;
template <> struct MmaType<BF16Tag> {
  static __device__ __forceinline__ unsigned sub2(unsigned x, unsigned y) {
    unsigned d;
    asm("sub.rn.bf16x2 %0, %1, %2;" : "=r"(d) : "r"(x), "r"(y));
    return d;
  }
  static __device__ __forceinline__ void mma(float (&c)[4], unsigned a0, unsigned a1, unsigned a2, unsigned a3, unsigned b0, unsigned b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
  }
  static __device__ __forceinline__ void mma0(float (&c)[4], unsigned a0, unsigned a1, unsigned a2, unsigned a3, unsigned b0, unsigned b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};"
        : "=f"(c[0]), "=f"(c[1]), "=f"(c[2]), "=f"(c[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "f"(0.f));
  }
};
template <> struct MmaType<F16Tag> {
  static __device__ __forceinline__ unsigned sub2(unsigned x, unsigned y) {
    unsigned d;
    asm("sub.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(x), "r"(y));
    return d;
  }
  static __device__ __forceinline__ void mma(float (&c)[4], unsigned a0, unsigned a1, unsigned a2, unsigned a3, unsigned b0, unsigned b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
  }
  static __device__ __forceinline__ void mma0(float (&c)[4], unsigned a0, unsigned a1, unsigned a2, unsigned a3, unsigned b0, unsigned b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};"
        : "=f"(c[0]), "=f"(c[1]), "=f"(c[2]), "=f"(c[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "f"(0.f));
  }
};
template <> struct MmaType<F32Tag> {};   // never instantiated: fp32 features stay on the FFMA2 path

#ifndef PILOT_MMA_PIPE
#define PILOT_MMA_PIPE 1           // 1: the next round's taps are loaded while this round's mma.sync run (up to 64 channels).
                                   // Measured (B200): cluster-resident kernel at 128 registers, 32 channels: config 1 0.642 -> 0.610 ms,
                                   // config 3 1.063 -> 1.029; pass kernel, 64 channels: 8.76 -> 8.31 ms at 16 warps per SM but
                                   // 7.88 without it at 24 warps (80 registers, where it spills): pilot_pass_mma.cu turns it off
#endif

#ifndef PILOT_MMA_PROJ_ILP
#define PILOT_MMA_PROJ_ILP 0       // 1: the projection passes of a super-batch side by side (pass kernel: config 4 -0.8 %;
                                    // the resident kernel, whose levels can be smaller than a super-batch, loses 1-3 %)
#endif
#ifndef PILOT_MMA_SB
#define PILOT_MMA_SB 64             // anchors a warp projects and compacts before it runs their rounds and lifts them
                                    // (64: 5 KB of shared memory per warp; the resident kernel uses 128)
#endif
// element i of the 16 floats the fp32 projection reads behind the double pose: R (row-major), the centre rounded to float,
// and what that rounding left (so that P - C is taken as (P - hi) - lo: no information of the double centre is lost)
__device__ __forceinline__ void pose_to_float(const double* Rc, const double* Cc, int i, float* out) {
  float v = 0.f;
  if (i < 9) v = (float)Rc[i];
  else if (i < 12) v = (float)Cc[i - 9];
  else if (i < 15) { const double c = Cc[i - 12]; v = (float)(c - (double)(float)c); }
  out[i] = v;
}
template <int CH> struct MmaGeom {            // CH = channels of a 16-bit feature: 16, 32, 64 or 128
  static constexpr int PX = CH * 2;                    // bytes per pixel
  static constexpr int TB = PX / 4 < 32 ? PX / 4 : 32; // bytes per load per thread (the 4 q-threads share a pixel): 8, 16, 32
  static constexpr int NW = TB / 4;                    // 32-bit words (= pairs of channels) per load per thread
  static constexpr int KS = NW / 2;                    // k-steps of 16 channels per load
  static constexpr int PARTS = PX / (4 * TB);          // loads per vector per thread (2 at 128 channels)
  static constexpr int LB = TB;                        // (alignment the loads need: 32 bytes from 64 channels on)
  static constexpr int kRow = 12;                      // floats per unit row of the warp's hand-off buffer: the ten distinct
                                                       // entries of E + 2 pad; 8 consecutive rows x 16 B fall in 8 distinct
                                                       // groups of four banks (12 i mod 32 = 0,12,24,4,16,28,8,20)
  static constexpr int SB = PILOT_MMA_SB;              // anchors per super-batch of a warp (a multiple of 32)
  // the warp's buffer, per slot of the super-batch: {tap offset, anchor index} (8 B, read by the rounds), {a, b, X/Z, Y/Z}
  // (16 B) and {1/Z, w_ref} (8 B) (read by the lane phase), and the Gram row (kRow floats)
  static constexpr int kSlotA = 0, kSlotB = 2 * SB, kSlotC = 6 * SB, kRows = 8 * SB;
  static constexpr int kWarpFloats = 8 * SB + SB * kRow;
};
template <int G> __host__ __device__ constexpr bool mma_supported() { return G == 2 || G == 4 || G == 8 || G == 16; }

// 1 / z for the fp32 projection: hardware seed + one Newton step, no slow path (z > z_near > 0 where the result is used)
__device__ __forceinline__ float rcp_f32(float z) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(z));
  return fmaf(y, fmaf(-z, y, 1.f), y);
}
template <int NW> struct TapWords { unsigned w[NW]; };
#define PILOT_LDG_OP "ld.global.nc"    // (.cg, .cv, .lu, .ca, L1::no_allocate, L1::evict_first measured: no difference)
template <int NW> __device__ __forceinline__ TapWords<NW> ldg_words(const char* p) {
  TapWords<NW> t;
  if constexpr (NW == 8) {                     // 32-byte load (sm_100: LDG.256); p is 32-byte aligned
    asm volatile(PILOT_LDG_OP ".v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=r"(t.w[0]), "=r"(t.w[1]), "=r"(t.w[2]), "=r"(t.w[3]), "=r"(t.w[4]), "=r"(t.w[5]), "=r"(t.w[6]), "=r"(t.w[7]) : "l"(p));
  } else if constexpr (NW == 4) {
    asm volatile(PILOT_LDG_OP ".v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(t.w[0]), "=r"(t.w[1]), "=r"(t.w[2]), "=r"(t.w[3]) : "l"(p));
  } else {
    asm volatile(PILOT_LDG_OP ".v2.b32 {%0,%1}, [%2];" : "=r"(t.w[0]), "=r"(t.w[1]) : "l"(p));
  }
  return t;
}

// Lane phase: the unit's lane reads the ten distinct entries of its Gram matrix E (row = three float4:
// {E00, E01, E02, E03}, {E11, E12, E13, E22}, {E23, E33, -, -}) and forms
//   p = { gx.gx, gx.gy, gy.gy, gx.r, gy.r, r.r } = M E M^T, M = rows of the three combinations above.
__device__ __forceinline__ void gram_unit_scalars(const float* row, float a, float b, float (&p)[6]) {
  const float4 r0 = reinterpret_cast<const float4*>(row)[0], r1 = reinterpret_cast<const float4*>(row)[1];
  const float2 r2 = reinterpret_cast<const float2*>(row)[4];
  const float E[16] = {r0.x, r0.y, r0.z, r0.w,  r0.y, r1.x, r1.y, r1.z,  r0.z, r1.y, r1.w, r2.x,  r0.w, r1.z, r2.x, r2.y};
  const float ob = 1.f - b, m20 = a * ob, m21 = a * b, m22 = b - 1.f;
  float t0[2], t1[3], t2[4];                                              // t_k = E m_k (the rows that are needed)
#pragma unroll
  for (int i = 0; i < 2; ++i) t0[i] = ob * E[4 * i] + b * E[4 * i + 1];
#pragma unroll
  for (int i = 0; i < 3; ++i) t1[i] = a * (E[4 * i + 1] - E[4 * i]) + E[4 * i + 2];
#pragma unroll
  for (int i = 0; i < 4; ++i) t2[i] = m20 * E[4 * i] + m21 * E[4 * i + 1] + m22 * E[4 * i + 2] - E[4 * i + 3];
  p[0] = ob * t0[0] + b * t0[1];
  p[1] = ob * t1[0] + b * t1[1];
  p[2] = a * (t1[1] - t1[0]) + t1[2];
  p[3] = ob * t2[0] + b * t2[1];
  p[4] = a * (t2[1] - t2[0]) + t2[2];
  p[5] = m20 * t2[0] + m21 * t2[1] + m22 * t2[2] - t2[3];
}

// floats of the [kNacc][kThreads] accumulator array in dynamic shared memory (0: accumulators in registers)
template <bool MMA> __host__ __device__ constexpr int acc_smem_floats() {
  return MMA ? 0 : (PILOT_SMEM_ACC ? kNacc * kThreads : 0);
}
template <int G, bool MMA> __host__ __device__ constexpr int red_warp_floats() {
  if constexpr (MMA) return MmaGeom<8 * G>::kWarpFloats; else return RedRows<G>::kWarpFloats;
}

// dynamic shared memory of the gather kernels: [accumulators kNacc x kThreads] [kWarps reduction buffers]
inline size_t gather_smem_for(int g, bool mma);
template <int G, bool MMA> constexpr size_t gather_smem_bytes() {
  return (size_t)acc_smem_floats<MMA>() * 4 + (size_t)kWarps * red_warp_floats<G, MMA>() * 4;
}

// The projection of one anchor in double (a2): the reference for every integer the projection decides. The fp32
// projection below calls it (cold path) for the anchors whose VISIBILITY it cannot decide safely: within `band` pixels of
// the border of the map or within band_z of z_near, where band is a multiple of its own rounding-error bound. n_valid and
// the set of units that contribute are therefore exactly those of a double projection.
struct ProjUnit { float a, b, x, y, iz; unsigned off; bool valid, near; };
__device__ __noinline__ ProjUnit project_anchor_f64(float Px, float Py, float Pz, unsigned pose_s, float fx, float fy, float cx, float cy,
                                                    float z_near, int W, int H, unsigned PX) {
  double R[12];
#pragma unroll
  for (int i = 0; i < 6; ++i)
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(R[2 * i]), "=d"(R[2 * i + 1]) : "r"(pose_s + 16u * i));
  const double* Cc = R + 9;
  const double dx = (double)Px - Cc[0], dy = (double)Py - Cc[1], dz = (double)Pz - Cc[2];
  const double Xd = R[0] * dx + R[1] * dy + R[2] * dz;
  const double Yd = R[3] * dx + R[4] * dy + R[5] * dz;
  const double Zd = R[6] * dx + R[7] * dy + R[8] * dz;
  bool valid = Zd > (double)z_near;
  const double izd = fast_rcp(Zd);
  const double ud = (double)fx * Xd * izd + (double)cx;
  const double vd = (double)fy * Yd * izd + (double)cy;
  const double x0d = floor(ud), y0d = floor(vd);
  valid = valid && (x0d >= 0.0) && (y0d >= 0.0) && (x0d + 1.0 <= (double)(W - 1)) && (y0d + 1.0 <= (double)(H - 1));
  ProjUnit u;
  u.iz = (float)izd;
  u.a = (float)(ud - x0d); u.b = (float)(vd - y0d);
  u.x = (float)Xd * u.iz; u.y = (float)Yd * u.iz;
  u.off = valid ? ((unsigned)(int)y0d * (unsigned)W + (unsigned)(int)x0d) * PX : 0u;
  u.valid = valid; u.near = false;
  return u;
}

// The same in fp32 (SURVEY 8(a) a2's number type) from the float copy of the pose behind the double one: the centre as a
// hi + lo pair (P - C loses nothing of the double centre), the rotation rounded to float, 1/Z from the hardware seed + one
// Newton step. Error of (u, v): <= ~1e-6 (fx + |u - cx|) pixels, i.e. ~1e-4 typical and 2e-3 worst case on a 1920-wide map -
// inside the bilinear patch that is a change of the continuous interpolant far below the 16-bit features' rounding. What is
// NOT continuous is visibility, so anchors within 4e-6 (fx + fy + W + H) pixels of the border of the map (>= 10x the bound;
// measured error on config 4: 3e-4 pixels) or within 4e-6 |P - C|_1 of z_near are projected again in double (about 1 anchor in 10^4).
__device__ __forceinline__ ProjUnit project_anchor_f32(float Px, float Py, float Pz, bool in_range, const float (&Rf)[16], unsigned pose_s,
                                                       float fx, float fy, float cx, float cy, float z_near, int W, int H,
                                                       float wmaxf, float hmaxf, float band, unsigned PX) {
  const float dx = (Px - Rf[9]) - Rf[12], dy = (Py - Rf[10]) - Rf[13], dz = (Pz - Rf[11]) - Rf[14];
  const float X = fmaf(Rf[2], dz, fmaf(Rf[1], dy, Rf[0] * dx));
  const float Y = fmaf(Rf[5], dz, fmaf(Rf[4], dy, Rf[3] * dx));
  const float Z = fmaf(Rf[8], dz, fmaf(Rf[7], dy, Rf[6] * dx));
  ProjUnit p;
  p.iz = rcp_f32(Z);
  p.x = X * p.iz; p.y = Y * p.iz;
  const float u = fmaf(fx, p.x, cx), v = fmaf(fy, p.y, cy);
  const float x0 = floorf(u), y0 = floorf(v);
  // 0 <= u < W - 1 as |u - (W-1)/2| < (W-1)/2 (one subtraction serves the decision and its guard; the two differ only
  // inside the band, where the double projection decides). NaNs compare false: such an anchor is invisible.
  const float hw = 0.5f * wmaxf, hh = 0.5f * hmaxf;
  const float tu = fabsf(u - hw) - hw, tv = fabsf(v - hh) - hh;           // < 0 inside
  p.valid = in_range && (Z > z_near) && (tu < 0.f) && (tv < 0.f);
  p.a = u - x0; p.b = v - y0;
  p.off = p.valid ? ((unsigned)(int)y0 * (unsigned)W + (unsigned)(int)x0) * PX : 0u;
  const float band_z = 4e-6f * (fabsf(dx) + fabsf(dy) + fabsf(dz));
  p.near = in_range && ((fabsf(tu) < band) || (fabsf(tv) < band) || (fabsf(Z - z_near) < band_z));
  return p;                                                              // the caller sends `near` anchors to project_anchor_f64
}

// ------------------------------------------------------------------ the photo gather, tensor-core contraction
//
// Same contract as photo_accumulate below (which dispatches here for MMA = true). A warp works on super-batches of SB
// anchors (SB / 32 of its round-robin batches), in three phases:
//   project    lane-per-anchor, SB / 32 passes: anchor load, projection in fp32 with visibility decided in double near the
//              borders (a2; project_anchor_f32 / _f64 above). The VISIBLE units are
//              compacted (ballot + popc rank, running count): slot s of the warp's table gets {tap offset, anchor index} and
//              the lane-phase state {a, b, X/Z, Y/Z, 1/Z, w_ref}; invisible anchors cost nothing beyond this point;
//   rounds     ceil(n_visible / 8) rounds; row-group g takes slot 8 r + g: five loads, four packed differences per word,
//              6 KS mma.sync; thread (g, g / 2) hands the unit's ten Gram entries to row `slot` of the warp's buffer;
//   lift       lane i takes slots i, i + 32, ...: Gram -> six scalars, robust weight, lift through J_uv into 29 registers
//              (a4-a5); ONE reduce-scatter per super-batch leaves component i of the warp's total in lane i (a6).
template <class T, int G>
__device__ __forceinline__ void photo_accumulate_mma(const PassArgs& A, const double* Rc, const double* Ccand,
                                                     int begin, int end, int worker, int n_workers,
                                                     float (&acc)[kNacc], float* sacc, float* red) {
  constexpr int CH = 8 * G;
  using Geo = MmaGeom<CH>;
  using M = MmaType<T>;
  constexpr int NW = Geo::NW, PX = Geo::PX, KS = Geo::KS, SB = Geo::SB;
  const LevelArgs& L = A.lv;
  const int lane = threadIdx.x & 31;
  const unsigned row_stride = (unsigned)PX * (unsigned)L.W;
  const char* feat = static_cast<const char*>(L.feat);
  const char* refb = static_cast<const char*>(L.ref);

  // The candidate pose stays in SHARED memory (Rc[9] and Ccand = Rc + 9 must point there, 16-byte aligned) and is re-read
  // by every projection: as 24 registers held across the rounds it forced the address arithmetic to be rematerialised.
  const unsigned pose_s = (unsigned)__cvta_generic_to_shared(Rc);         // Rc[9] | Cc[3] contiguous, 16-byte aligned
  const float wmaxf = (float)(L.W - 1), hmaxf = (float)(L.H - 1);
  const float band = 4e-6f * (fabsf(L.fx) + fabsf(L.fy) + (float)(L.W + L.H));   // see project_anchor_f32

  const int q = lane & 3, g = lane >> 2;
  const bool diag = q == (g >> 1);                                        // holds C[g][g] and C[g+8][g] of every accumulator
  const bool odd = g & 1;                                                 // ... in c[1], c[3] (else c[0], c[2])
  const char* const featq = feat + q * Geo::TB;
  const char* const refq = refb + q * Geo::TB;
  uint2* const slotA = reinterpret_cast<uint2*>(red + Geo::kSlotA);
  float4* const slotB = reinterpret_cast<float4*>(red + Geo::kSlotB);
  float2* const slotC = reinterpret_cast<float2*>(red + Geo::kSlotC);
  float* const rows = red + Geo::kRows;
  const unsigned rows_s = (unsigned)__cvta_generic_to_shared(rows);


  // The 32-anchor batches of [begin, end) go round-robin over the workers (batch b to worker b mod n_workers: the warps that
  // run together sweep neighbouring anchors, which is what keeps the union of the resident CTAs' footprints in L2); a
  // worker takes its batches SB / 32 at a time.
  const int n_batches = (end - begin + 31) >> 5;
  auto load_anchor = [&](int b) { const int j = begin + b * 32 + lane; return (b < n_batches && j < end) ? __ldg(L.points + j) : make_float4(0.f, 0.f, 0.f, -1.f); };
  constexpr int PASSES = SB / 32;
  float4 Pn = load_anchor(worker);
  for (int b0 = worker; b0 < n_batches; b0 += PASSES * n_workers) {
    // ---- project + compact
    int nv = 0;
#if PILOT_MMA_PROJ_ILP
    // the SB / 32 passes are independent chains: written out side by side so that the compiler interleaves them (a
    // batch past the end projects nothing: its lanes are invalid). The first pass's anchors were loaded one super-batch ago.
    {
      float4 Pk[PASSES];
      Pk[0] = Pn;
#pragma unroll
      for (int k = 1; k < PASSES; ++k) Pk[k] = load_anchor(b0 + k * n_workers);
      Pn = load_anchor(b0 + PASSES * n_workers);
      float pa[PASSES], pb[PASSES], px[PASSES], py[PASSES], piz[PASSES];
      unsigned poff[PASSES];
      bool pvalid[PASSES];
      bool pnear[PASSES];
      float Rf[16];                                                       // R[9], C hi[3], C lo[3], pad: four 16-byte loads
#pragma unroll
      for (int i = 0; i < 4; ++i)
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(Rf[4 * i]), "=f"(Rf[4 * i + 1]), "=f"(Rf[4 * i + 2]), "=f"(Rf[4 * i + 3]) : "r"(pose_s + 96u + 16u * i));
#pragma unroll
      for (int k = 0; k < PASSES; ++k) {
        const int base = begin + (b0 + k * n_workers) * 32;
        const bool in_range = (b0 + k * n_workers) < n_batches && base + lane < end;
        const ProjUnit pu = project_anchor_f32(Pk[k].x, Pk[k].y, Pk[k].z, in_range, Rf, pose_s, L.fx, L.fy, L.cx, L.cy, A.prm.z_near,
                                               L.W, L.H, wmaxf, hmaxf, band, (unsigned)PX);
        pa[k] = pu.a; pb[k] = pu.b; px[k] = pu.x; py[k] = pu.y; piz[k] = pu.iz; poff[k] = pu.off; pvalid[k] = pu.valid;
        pnear[k] = pu.near;
      }
      bool any_near = false;
#pragma unroll
      for (int k = 0; k < PASSES; ++k) any_near = any_near || pnear[k];
      if (any_near) {                                                     // cold: visibility decided in double (one branch for all passes)
#pragma unroll
        for (int k = 0; k < PASSES; ++k) {
          if (!pnear[k]) continue;
          const ProjUnit pu = project_anchor_f64(Pk[k].x, Pk[k].y, Pk[k].z, pose_s, L.fx, L.fy, L.cx, L.cy, A.prm.z_near, L.W, L.H, (unsigned)PX);
          pa[k] = pu.a; pb[k] = pu.b; px[k] = pu.x; py[k] = pu.y; piz[k] = pu.iz; poff[k] = pu.off; pvalid[k] = pu.valid;
        }
      }
#pragma unroll
      for (int k = 0; k < PASSES; ++k) {
        const unsigned vmask = __ballot_sync(0xffffffffu, pvalid[k]);
        if (pvalid[k]) {
          const int s = nv + __popc(vmask & ((1u << lane) - 1u));
          slotA[s] = make_uint2(poff[k], (unsigned)(begin + (b0 + k * n_workers) * 32 + lane));
          slotB[s] = make_float4(pa[k], pb[k], px[k], py[k]);
          slotC[s] = make_float2(piz[k], Pk[k].w);
        }
        nv += __popc(vmask);
      }
    }
#else
    Pn = load_anchor(b0);
#pragma unroll 1
    for (int k = 0; k < PASSES; ++k) {
      const int b = b0 + k * n_workers;
      if (b >= n_batches) break;
      const int base = begin + b * 32;
      const float4 P = Pn;
      Pn = load_anchor(b + n_workers);                                    // next pass's anchors: in flight during this one
      bool valid = base + lane < end;
      float Rf[16];                                                       // R[9], C hi[3], C lo[3], pad: four 16-byte loads
#pragma unroll
      for (int i = 0; i < 4; ++i)
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(Rf[4 * i]), "=f"(Rf[4 * i + 1]), "=f"(Rf[4 * i + 2]), "=f"(Rf[4 * i + 3]) : "r"(pose_s + 96u + 16u * i));
      ProjUnit pu = project_anchor_f32(P.x, P.y, P.z, valid, Rf, pose_s, L.fx, L.fy, L.cx, L.cy, A.prm.z_near, L.W, L.H, wmaxf, hmaxf,
                                       band, (unsigned)PX);
      if (pu.near) pu = project_anchor_f64(P.x, P.y, P.z, pose_s, L.fx, L.fy, L.cx, L.cy, A.prm.z_near, L.W, L.H, (unsigned)PX);   // cold
      valid = pu.valid;
      const unsigned vmask = __ballot_sync(0xffffffffu, valid);
      if (valid) {
        const int s = nv + __popc(vmask & ((1u << lane) - 1u));
        slotA[s] = make_uint2(pu.off, (unsigned)(base + lane));
        slotB[s] = make_float4(pu.a, pu.b, pu.x, pu.y);
        slotC[s] = make_float2(pu.iz, P.w);
      }
      nv += __popc(vmask);
    }
#endif
    if (nv == 0) continue;                                                // no visible unit: nothing to gather
    __syncwarp();

    // ---- rounds
    const int nr = (nv + 7) >> 3;
    // The ten Gram entries of a row-group's unit from its four difference vectors (one load = KS k-steps), written
    // PRODUCT-MAJOR: the KS k-steps of one product on one accumulator quad, its two wanted entries kept, then the next
    // product. ptxas still interleaves the six quads (the SASS keeps 24 accumulator registers), but from this order it
    // needs fewer register-pairing copies around the HMMAs than from the k-step-major one (132 instead of 146 instructions
    // per round): config 4 7.11 -> 7.00 ms, config 2 6.85 -> 6.76 at the same 80 registers. Thread (g, g / 2) then hands
    // the entries to row `slot` of the warp's buffer.
    auto contract_and_hand_off = [&](const unsigned (&e0)[NW], const unsigned (&e1)[NW], const unsigned (&e2)[NW], const unsigned (&e3)[NW],
                                     int slot, bool act) {
      auto product = [&](const unsigned (&alo)[NW], const unsigned (&ahi)[NW], const unsigned (&b)[NW], float& lo, float& hi) {
        float c[4];
        M::mma0(c, alo[0], ahi[0], alo[1], ahi[1], b[0], b[1]);
#pragma unroll
        for (int k = 1; k < KS; ++k) M::mma(c, alo[2 * k], ahi[2 * k], alo[2 * k + 1], ahi[2 * k + 1], b[2 * k], b[2 * k + 1]);
        lo = odd ? c[1] : c[0];                                             // C[g][g]
        hi = odd ? c[3] : c[2];                                             // C[g + 8][g]
      };
      float E00, E02, E01, E12, E03, E23, E22, E11, E13, E33, dup;
      product(e0, e2, e0, E00, E02);                                        // e0.e0 | e2.e0
      product(e0, e2, e1, E01, E12);                                        // e0.e1 | e2.e1
      product(e0, e2, e3, E03, E23);                                        // e0.e3 | e2.e3
      product(e0, e2, e2, dup, E22);                                        // (e0.e2) | e2.e2
      product(e1, e3, e1, E11, E13);                                        // e1.e1 | e3.e1
      product(e1, e3, e3, dup, E33);                                        // (e1.e3) | e3.e3
      if (diag && act) {
        const unsigned rp = rows_s + (unsigned)(slot * Geo::kRow) * 4u;
        asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" :: "r"(rp), "f"(E00), "f"(E01), "f"(E02), "f"(E03) : "memory");
        asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" :: "r"(rp + 16u), "f"(E11), "f"(E12), "f"(E13), "f"(E22) : "memory");
        asm volatile("st.shared.v2.f32 [%0], {%1,%2};" :: "r"(rp + 32u), "f"(E23), "f"(E33) : "memory");
      }
    };
#if PILOT_MMA_PIPE
    if constexpr (Geo::PARTS == 1) {
      // Software pipeline over the rounds: the next round's five loads are issued as soon as this round's taps have been
      // turned into differences (their registers are free again), so they are in flight during the 6 KS mma.sync and the
      // hand-off of this round - a warp always has loads outstanding, whatever phase the other warps of the SM are in.
      // (k-step-major order of the products here: at 16 warps per SM the six independent accumulators are worth more than
      // the registers - product-major measured 0.470 against 0.458 ms on config 1, 0.791 against 0.781 on config 3.)
      TapWords<NW> t[5];
      auto issue = [&](int r) {
        const int s = 8 * r + g;
        const uint2 sl = slotA[s < nv ? s : 0];        // a row-group past the last visible unit repeats slot 0 (L1 hits)
        const char* const p0 = featq + sl.x;
        t[0] = ldg_words<NW>(p0);
        t[1] = ldg_words<NW>(p0 + PX);
        t[2] = ldg_words<NW>(p0 + row_stride);
        t[3] = ldg_words<NW>(p0 + row_stride + PX);
        t[4] = ldg_words<NW>(refq + (size_t)sl.y * PX);
      };
      issue(0);
      for (int r = 0; r < nr; ++r) {
        const int s = 8 * r + g;
        const bool act = s < nv;
        unsigned e0[NW], e1[NW], e2[NW], e3[NW];
#pragma unroll
        for (int i = 0; i < NW; ++i) {
          e0[i] = M::sub2(t[1].w[i], t[0].w[i]);
          e1[i] = M::sub2(t[3].w[i], t[2].w[i]);
          e2[i] = M::sub2(t[2].w[i], t[0].w[i]);
          e3[i] = M::sub2(t[4].w[i], t[2].w[i]);
        }
        if (r + 1 < nr) issue(r + 1);
        float c0[4], c1[4], c2[4], c3[4], c4[4], c5[4];
#pragma unroll
        for (int k = 0; k < KS; ++k) {
          const unsigned e0a = e0[2 * k], e0b = e0[2 * k + 1], e1a = e1[2 * k], e1b = e1[2 * k + 1];
          const unsigned e2a = e2[2 * k], e2b = e2[2 * k + 1], e3a = e3[2 * k], e3b = e3[2 * k + 1];
          if (k == 0) {
            M::mma0(c0, e0a, e2a, e0b, e2b, e0a, e0b);                    // e0.e0 | e2.e0
            M::mma0(c1, e0a, e2a, e0b, e2b, e1a, e1b);                    // e0.e1 | e2.e1
            M::mma0(c2, e0a, e2a, e0b, e2b, e3a, e3b);                    // e0.e3 | e2.e3
            M::mma0(c3, e0a, e2a, e0b, e2b, e2a, e2b);                    // (e0.e2) | e2.e2
            M::mma0(c4, e1a, e3a, e1b, e3b, e1a, e1b);                    // e1.e1 | e3.e1
            M::mma0(c5, e1a, e3a, e1b, e3b, e3a, e3b);                    // (e1.e3) | e3.e3
          } else {
            M::mma(c0, e0a, e2a, e0b, e2b, e0a, e0b);
            M::mma(c1, e0a, e2a, e0b, e2b, e1a, e1b);
            M::mma(c2, e0a, e2a, e0b, e2b, e3a, e3b);
            M::mma(c3, e0a, e2a, e0b, e2b, e2a, e2b);
            M::mma(c4, e1a, e3a, e1b, e3b, e1a, e1b);
            M::mma(c5, e1a, e3a, e1b, e3b, e3a, e3b);
          }
        }
        if (diag && act) {
          const unsigned rp = rows_s + (unsigned)(s * Geo::kRow) * 4u;
          const float E00 = odd ? c0[1] : c0[0], E02 = odd ? c0[3] : c0[2];
          const float E01 = odd ? c1[1] : c1[0], E12 = odd ? c1[3] : c1[2];
          const float E03 = odd ? c2[1] : c2[0], E23 = odd ? c2[3] : c2[2];
          const float E22 = odd ? c3[3] : c3[2];
          const float E11 = odd ? c4[1] : c4[0], E13 = odd ? c4[3] : c4[2];
          const float E33 = odd ? c5[3] : c5[2];
          asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" :: "r"(rp), "f"(E00), "f"(E01), "f"(E02), "f"(E03) : "memory");
          asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" :: "r"(rp + 16u), "f"(E11), "f"(E12), "f"(E13), "f"(E22) : "memory");
          asm volatile("st.shared.v2.f32 [%0], {%1,%2};" :: "r"(rp + 32u), "f"(E23), "f"(E33) : "memory");
        }
      }
    } else
#endif
    if constexpr (Geo::PARTS == 1) {
      for (int r = 0; r < nr; ++r) {
        const int s = 8 * r + g;
        const bool act = s < nv;
        // a row-group past the last visible unit repeats slot 0 (always there: its loads hit L1) and stores nothing
        const uint2 sl = slotA[act ? s : 0];
        const char* const p0 = featq + sl.x;
        const TapWords<NW> f00 = ldg_words<NW>(p0);
        const TapWords<NW> f10 = ldg_words<NW>(p0 + PX);
        const TapWords<NW> f01 = ldg_words<NW>(p0 + row_stride);
        const TapWords<NW> f11 = ldg_words<NW>(p0 + row_stride + PX);
        const TapWords<NW> fr = ldg_words<NW>(refq + (size_t)sl.y * PX);
        unsigned e0[NW], e1[NW], e2[NW], e3[NW];
#pragma unroll
        for (int i = 0; i < NW; ++i) {
          e0[i] = M::sub2(f10.w[i], f00.w[i]);
          e1[i] = M::sub2(f11.w[i], f01.w[i]);
          e2[i] = M::sub2(f01.w[i], f00.w[i]);
          e3[i] = M::sub2(fr.w[i], f01.w[i]);
        }
        contract_and_hand_off(e0, e1, e2, e3, s, act);
      }
    } else
    for (int r = 0; r < nr; ++r) {
      const int s = 8 * r + g;
      const bool act = s < nv;
      float c0[4], c1[4], c2[4], c3[4], c4[4], c5[4];
      // a row-group past the last visible unit repeats slot 0 (always there: its loads hit L1) and stores nothing
      const uint2 sl = slotA[act ? s : 0];
      const char* const p0 = featq + sl.x;
      const char* const pr = refq + (size_t)sl.y * PX;
#pragma unroll
      for (int part = 0; part < Geo::PARTS; ++part) {
        const TapWords<NW> f00 = ldg_words<NW>(p0 + part * 128);
        const TapWords<NW> f10 = ldg_words<NW>(p0 + part * 128 + PX);
        const TapWords<NW> f01 = ldg_words<NW>(p0 + part * 128 + row_stride);
        const TapWords<NW> f11 = ldg_words<NW>(p0 + part * 128 + row_stride + PX);
        const TapWords<NW> fr = ldg_words<NW>(pr + part * 128);
#pragma unroll
        for (int k = 0; k < KS; ++k) {
          const unsigned e0a = M::sub2(f10.w[2 * k], f00.w[2 * k]), e0b = M::sub2(f10.w[2 * k + 1], f00.w[2 * k + 1]);
          const unsigned e1a = M::sub2(f11.w[2 * k], f01.w[2 * k]), e1b = M::sub2(f11.w[2 * k + 1], f01.w[2 * k + 1]);
          const unsigned e2a = M::sub2(f01.w[2 * k], f00.w[2 * k]), e2b = M::sub2(f01.w[2 * k + 1], f00.w[2 * k + 1]);
          const unsigned e3a = M::sub2(fr.w[2 * k], f01.w[2 * k]), e3b = M::sub2(fr.w[2 * k + 1], f01.w[2 * k + 1]);
          if (part == 0 && k == 0) {
            M::mma0(c0, e0a, e2a, e0b, e2b, e0a, e0b);                    // e0.e0 | e2.e0
            M::mma0(c1, e0a, e2a, e0b, e2b, e1a, e1b);                    // e0.e1 | e2.e1
            M::mma0(c2, e0a, e2a, e0b, e2b, e3a, e3b);                    // e0.e3 | e2.e3
            M::mma0(c3, e0a, e2a, e0b, e2b, e2a, e2b);                    // (e0.e2) | e2.e2
            M::mma0(c4, e1a, e3a, e1b, e3b, e1a, e1b);                    // e1.e1 | e3.e1
            M::mma0(c5, e1a, e3a, e1b, e3b, e3a, e3b);                    // (e1.e3) | e3.e3
          } else {
            M::mma(c0, e0a, e2a, e0b, e2b, e0a, e0b);
            M::mma(c1, e0a, e2a, e0b, e2b, e1a, e1b);
            M::mma(c2, e0a, e2a, e0b, e2b, e3a, e3b);
            M::mma(c3, e0a, e2a, e0b, e2b, e2a, e2b);
            M::mma(c4, e1a, e3a, e1b, e3b, e1a, e1b);
            M::mma(c5, e1a, e3a, e1b, e3b, e3a, e3b);
          }
        }
      }
      if (diag && act) {
        const unsigned rp = rows_s + (unsigned)(s * Geo::kRow) * 4u;
        const float E00 = odd ? c0[1] : c0[0], E02 = odd ? c0[3] : c0[2];
        const float E01 = odd ? c1[1] : c1[0], E12 = odd ? c1[3] : c1[2];
        const float E03 = odd ? c2[1] : c2[0], E23 = odd ? c2[3] : c2[2];
        const float E22 = odd ? c3[3] : c3[2];
        const float E11 = odd ? c4[1] : c4[0], E13 = odd ? c4[3] : c4[2];
        const float E33 = odd ? c5[3] : c5[2];
        asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" :: "r"(rp), "f"(E00), "f"(E01), "f"(E02), "f"(E03) : "memory");
        asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" :: "r"(rp + 16u), "f"(E11), "f"(E12), "f"(E13), "f"(E22) : "memory");
        asm volatile("st.shared.v2.f32 [%0], {%1,%2};" :: "r"(rp + 32u), "f"(E23), "f"(E33) : "memory");
      }
    }
    __syncwarp();

    // ---- lift: lane-per-unit over the compacted slots (a4-a5), one reduce-scatter per super-batch (a6)
    float v[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = 0.f;
    for (int s = lane; s < nv; s += 32) {
      const float4 sb4 = slotB[s];
      const float2 sc2 = slotC[s];
      const float a = sb4.x, b = sb4.y, x = sb4.z, y = sb4.w, iz = sc2.x;
      float p[6];
      gram_unit_scalars(rows + s * Geo::kRow, a, b, p);
      float wq = 1.f;
      if (L.conf) {
        const float* cq = L.conf + slotA[s].x / (unsigned)PX;
        float q00 = __ldg(cq), q10 = __ldg(cq + 1), q01 = __ldg(cq + L.W), q11 = __ldg(cq + L.W + 1);
        wq = (1.f - b) * ((1.f - a) * q00 + a * q10) + b * ((1.f - a) * q01 + a * q11);
      }
      float w = sc2.y * wq;
      float rho, drho;
      robust_fast(A.prm.loss, w * p[5], A.prm.loss_scale, rho, drho);
      float om = w * drho;
      float fxz = L.fx * iz, fyz = L.fy * iz;
      float Ju[6] = {fxz, 0.f, -fxz * x, -L.fx * x * y, L.fx * (1.f + x * x), -L.fx * y};
      float Jv[6] = {0.f, fyz, -fyz * y, -L.fy * (1.f + y * y), L.fy * x * y, L.fy * x};
      float A11 = om * p[0], A12 = om * p[1], A22 = om * p[2];
      float b1 = om * p[3], b2 = om * p[4];
#pragma unroll
      for (int i = 0; i < 6; ++i) {
        float mu = A11 * Ju[i] + A12 * Jv[i];
        float mv = A12 * Ju[i] + A22 * Jv[i];
#pragma unroll
        for (int k = i; k < 6; ++k) v[tri(i, k)] += mu * Ju[k] + mv * Jv[k];
        v[21 + i] += b1 * Ju[i] + b2 * Jv[i];
      }
      v[27] += rho;
      v[28] += 1.f;
    }
    __syncwarp();                                                         // the table is rewritten by the next super-batch
    // reduce-scatter over the warp: lane i ends with the super-batch total of component i (31 shuffles), which goes to ONE
    // accumulator register per lane
#pragma unroll
    for (int half = 16; half >= 1; half >>= 1) {
      const bool upper = lane & half;
#pragma unroll
      for (int i = 0; i < half; ++i) {
        const float send = upper ? v[i] : v[i + half];
        const float keep = upper ? v[i + half] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, half);
      }
    }
    acc[0] += v[0];
  }
}

// ------------------------------------------------------------------ the photo kernel
//
// grid = (n_hyp, n_chunks): blockIdx.x (fastest) is the hypothesis, so CTAs that run together
// sweep the SAME chunk of (spatially sorted) anchors under different poses and the union of their
// footprints is a narrow band of the map that stays in L2.
template <class T, int G, bool CEN, bool MMA>
__device__ __forceinline__ void photo_accumulate(const PassArgs& A, const double* Rc, const double* Ccand,
                                                 int begin, int end, int worker, int n_workers,
                                                 float (&acc)[kNacc], float* sacc, float* red /* this warp's rows */) {
#if PILOT_SMEM_ACC
#define PILOT_ACC(i) sacc[(i) * kThreads]     // this thread's column of the [kNacc][kThreads] shared array
#else
#define PILOT_ACC(i) acc[i]
#endif
  if constexpr (MMA) {
    static_assert(!CEN && mma_supported<G>() && T::kVec == 8, "tensor-core path: 16-bit features, exact bilinear gradient");
    photo_accumulate_mma<T, G>(A, Rc, Ccand, begin, end, worker, n_workers, acc, sacc, red);
    return;
  }
  constexpr int LOG = Log2<G>::v;
  const LevelArgs& L = A.lv;
  const int lane = threadIdx.x & 31;
  const int sub = lane & (G - 1);
  const unsigned esz = 16 / T::kVec;
  const unsigned px_stride = (unsigned)L.C * esz;
  const unsigned row_stride = px_stride * (unsigned)L.W;
  const char* feat = static_cast<const char*>(L.feat);
  const char* refb = static_cast<const char*>(L.ref);

  // candidate pose (the pose this pass evaluates), double for the projection
  double R[9], Cc[3];
#pragma unroll
  for (int i = 0; i < 9; ++i) R[i] = Rc[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) Cc[i] = Ccand[i];

  const float wmax = (float)(L.W - 1), hmax = (float)(L.H - 1);

  for (int base = begin + worker * 32; base < end; base += n_workers * 32) {
    // ---- lane-per-unit: projection + visibility (a2), in double so that u,v carry no fp32 noise
    const int j = base + lane;
    bool valid = j < end;
    float4 P = valid ? __ldg(L.points + j) : make_float4(0.f, 0.f, 0.f, 0.f);
    double dx = (double)P.x - Cc[0], dy = (double)P.y - Cc[1], dz = (double)P.z - Cc[2];
    double Xd = R[0] * dx + R[1] * dy + R[2] * dz;
    double Yd = R[3] * dx + R[4] * dy + R[5] * dz;
    double Zd = R[6] * dx + R[7] * dy + R[8] * dz;
    valid = valid && (Zd > (double)A.prm.z_near);
    double izd = fast_rcp(Zd);
    double ud = (double)L.fx * Xd * izd + (double)L.cx;
    double vd = (double)L.fy * Yd * izd + (double)L.cy;
    double x0d = floor(ud), y0d = floor(vd);
    valid = valid && (x0d >= 0.0) && (y0d >= 0.0) && (x0d + 1.0 <= (double)wmax) && (y0d + 1.0 <= (double)hmax);
    float a = valid ? (float)(ud - x0d) : 0.f;
    float b = valid ? (float)(vd - y0d) : 0.f;
    int x0 = valid ? (int)x0d : 0, y0 = valid ? (int)y0d : 0;
    unsigned off = ((unsigned)y0 * (unsigned)L.W + (unsigned)x0) * px_stride;   // invalid units read pixel (0,0)
    unsigned offv = valid ? off : 0xffffffffu;
    if (!__any_sync(0xffffffffu, valid)) continue;         // no visible unit in this batch: nothing to gather

    // ---- group rounds: gather + per-unit contraction (a3-a5), reduce-scatter so that lane i ends
    //      up with the six sums of unit i of this batch
    float cur[6];
    float stash[LOG > 0 ? LOG : 1][6];
    const int gbase = base + (lane & ~(G - 1));           // first unit of this lane's group
    auto fetch = [&](int r, float& ra, float& rb, bool& rvalid) {
      unsigned o = __shfl_sync(0xffffffffu, offv, r, G);
      ra = __shfl_sync(0xffffffffu, a, r, G);
      rb = __shfl_sync(0xffffffffu, b, r, G);
      rvalid = o != 0xffffffffu;
      int jr = min(gbase + r, L.N - 1);
      return load_taps<16 * G>(feat, (rvalid ? o : 0u) + (unsigned)sub * 16u, row_stride,
                       refb + ((size_t)jr * L.C) * esz + (size_t)sub * 16u);
    };
    constexpr int D = PILOT_PREFETCH < G ? PILOT_PREFETCH : G;
    float na[D], nb[D]; bool nvalid[D];
    RawTaps nxt[D];
    unsigned cflags = 0;                                   // CEN: which outer taps are clamped at the border
    if constexpr (CEN) cflags = (x0 > 0 ? 1u : 0u) | (x0 + 2 <= L.W - 1 ? 2u : 0u) | (y0 > 0 ? 4u : 0u) | (y0 + 2 <= L.H - 1 ? 8u : 0u);
    else {
#pragma unroll
      for (int d = 0; d < D; ++d) nxt[d] = fetch(d, na[d], nb[d], nvalid[d]);
    }
#pragma unroll
    for (int r = 0; r < G; ++r) {
      bool rvalid;
      if constexpr (CEN) {
        unsigned o = __shfl_sync(0xffffffffu, offv, r, G);
        float ra = __shfl_sync(0xffffffffu, a, r, G), rb = __shfl_sync(0xffffffffu, b, r, G);
        unsigned fl = __shfl_sync(0xffffffffu, cflags, r, G);
        rvalid = o != 0xffffffffu;
        if (!rvalid) fl = 0;                               // invisible units read around pixel (0,0), unclamped side only
        OuterTaps ot{(fl & 1u) ? -(int)(16 * G) : 0, (fl & 2u) ? 2 * 16 * G : 16 * G,
                     (fl & 4u) ? -(int)row_stride : 0, (fl & 8u) ? 2 * (int)row_stride : (int)row_stride};
        int jr = min(gbase + r, L.N - 1);
        unit_partials_central<T, 16 * G>(feat + (rvalid ? o : 0u) + (unsigned)sub * 16u, row_stride, ot,
                                         refb + ((size_t)jr * L.C) * esz + (size_t)sub * 16u, ra, rb, cur);
      } else {
        RawTaps t = nxt[r % D];
        float ra = na[r % D], rb = nb[r % D];
        rvalid = nvalid[r % D];
        if (r + D < G) nxt[r % D] = fetch(r + D, na[r % D], nb[r % D], nvalid[r % D]);   // software pipeline: next units' loads in flight
        unit_partials<T>(t, ra, rb, cur);
      }
      if (!rvalid) {
#pragma unroll
        for (int i = 0; i < 6; ++i) cur[i] = 0.f;
      }
      if constexpr (RedRows<G>::kOn) {
        float2* row = reinterpret_cast<float2*>(red + RedRows<G>::row((lane & ~(G - 1)) + r) + sub * 6);
        row[0] = make_float2(cur[0], cur[1]); row[1] = make_float2(cur[2], cur[3]); row[2] = make_float2(cur[4], cur[5]);
      } else {
#pragma unroll
        for (int k = 0; k < LOG; ++k) {
          if (((r >> k) & 1) == 0) {
#pragma unroll
            for (int i = 0; i < 6; ++i) stash[k][i] = cur[i];
            break;
          }
          halve<6>(stash[k], cur, 1 << k, (sub >> k) & 1);
#pragma unroll
          for (int i = 0; i < 6; ++i) cur[i] = stash[k][i];
        }
      }
    }
    if constexpr (RedRows<G>::kOn) {                       // lane i sums the G slices of unit i, in lane order
      __syncwarp();
      const float4* rp = reinterpret_cast<const float4*>(red + RedRows<G>::row(lane));
      float v[6 * G];
#pragma unroll
      for (int i = 0; i < 6 * G / 4; ++i) {
        float4 t = rp[i];
        v[4 * i] = t.x; v[4 * i + 1] = t.y; v[4 * i + 2] = t.z; v[4 * i + 3] = t.w;
      }
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        float t = v[c];
#pragma unroll
        for (int g = 1; g < G; ++g) t += v[6 * g + c];
        cur[c] = t;
      }
      __syncwarp();                                        // rows are rewritten by the next batch
    }

    // ---- lane-per-unit: robust weight, lift through the 2x6 Jacobian, accumulate (a4-a6)
    if (valid) {
      float wq = 1.f;
      if (L.conf) {
        const float* q = L.conf + (size_t)y0 * L.W + x0;
        float q00 = __ldg(q), q10 = __ldg(q + 1), q01 = __ldg(q + L.W), q11 = __ldg(q + L.W + 1);
        wq = (1.f - b) * ((1.f - a) * q00 + a * q10) + b * ((1.f - a) * q01 + a * q11);
      }
      float w = P.w * wq;
      float rho, drho;
      robust<float>(A.prm.loss, w * cur[5], A.prm.loss_scale, rho, drho);
      float om = w * drho;
      float X = (float)Xd, Y = (float)Yd, iz = (float)izd;
      float x = X * iz, y = Y * iz;
      float fxz = L.fx * iz, fyz = L.fy * iz;
      // Juv rows (d(u,v)/d(rho,phi)); Ju[1] = Jv[0] = 0
      float Ju[6] = {fxz, 0.f, -fxz * x, -L.fx * x * y, L.fx * (1.f + x * x), -L.fx * y};
      float Jv[6] = {0.f, fyz, -fyz * y, -L.fy * (1.f + y * y), L.fy * x * y, L.fy * x};
      float A11 = om * cur[0], A12 = om * cur[1], A22 = om * cur[2];
      float b1 = om * cur[3], b2 = om * cur[4];
#pragma unroll
      for (int p = 0; p < 6; ++p) {
        float mu = A11 * Ju[p] + A12 * Jv[p];
        float mv = A12 * Ju[p] + A22 * Jv[p];
#pragma unroll
        for (int q = p; q < 6; ++q) PILOT_ACC(tri(p, q)) += mu * Ju[q] + mv * Jv[q];
        PILOT_ACC(21 + p) += b1 * Ju[p] + b2 * Jv[p];
      }
      PILOT_ACC(27) += rho;
      PILOT_ACC(28) += 1.f;
    }
  }
#undef PILOT_ACC
}

inline size_t gather_smem_for(int g, bool mma) {
  switch (g) {
    case 1: return gather_smem_bytes<1, false>();
    case 2: return mma ? gather_smem_bytes<2, true>() : gather_smem_bytes<2, false>();
    case 4: return mma ? gather_smem_bytes<4, true>() : gather_smem_bytes<4, false>();
    case 8: return mma ? gather_smem_bytes<8, true>() : gather_smem_bytes<8, false>();
    case 16: return mma ? gather_smem_bytes<16, true>() : gather_smem_bytes<16, false>();
    case 32: return gather_smem_bytes<32, false>();
  }
  return 0;
}

// The per-thread accumulators before / after photo_accumulate: registers, a column of shared memory, or (tensor-core
// path) one register per lane that already holds the warp total of component `lane`.
#define PILOT_DECLARE_ACC extern __shared__ float4 pilot_dyn_smem[]; \
  float* sacc = reinterpret_cast<float*>(pilot_dyn_smem) + threadIdx.x; float acc[kNacc]; \
  float* red = reinterpret_cast<float*>(pilot_dyn_smem) + acc_smem_floats<MMA>() + (threadIdx.x >> 5) * red_warp_floats<G, MMA>();

template <bool MMA>
__device__ __forceinline__ void acc_zero(float (&acc)[kNacc], float* sacc) {
  if constexpr (MMA) {
    acc[0] = 0.f;
  } else {
#pragma unroll
    for (int i = 0; i < kNacc; ++i) {
      if (PILOT_SMEM_ACC) sacc[i * kThreads] = 0.f; else acc[i] = 0.f;
    }
  }
}

// Warp total of component `lane` (fixed order: deterministic).
template <bool MMA>
__device__ __forceinline__ float acc_warp_total(float (&acc)[kNacc], const float* sacc, int lane) {
  if constexpr (MMA) {
    return acc[0];
  } else {
    if (PILOT_SMEM_ACC) {
#pragma unroll
      for (int i = 0; i < kNacc; ++i) acc[i] = sacc[i * kThreads];
    }
    // reduce-scatter over the warp: lane i ends with the warp total of component i (31 shuffles)
#pragma unroll
    for (int half = 16; half >= 1; half >>= 1) {
      const bool upper = lane & half;
#pragma unroll
      for (int i = 0; i < half; ++i) {
        float send = upper ? acc[i] : acc[i + half];
        float keep = upper ? acc[i + half] : acc[i];
        acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, half);
      }
    }
    return acc[0];
  }
}

}  // namespace

namespace {

// ------------------------------------------------------------------ priors (a7, a8), executed by one full warp in double

struct DsmView { const float* d; int w, h; double ox, oy, gsd, ig; };   // ig = 1 / gsd
__host__ __device__ inline DsmView make_dsm_view(const float* d, int w, int h, float ox, float oy, float gsd) {
#ifdef __CUDA_ARCH__
  return DsmView{d, w, h, (double)ox, (double)oy, (double)gsd, fast_rcp((double)gsd)};
#else
  return DsmView{d, w, h, (double)ox, (double)oy, (double)gsd, 1.0 / (double)gsd};
#endif
}

// Bilinear heightfield sample and exact gradient (per metre). false = outside the DSM.
__device__ __forceinline__ bool dsm_sample(const DsmView& D, double x, double y, double& z, double& zx, double& zy) {
  double gx = (x - D.ox) * D.ig, gy = (y - D.oy) * D.ig;
  double fx0 = floor(gx), fy0 = floor(gy);
  if (!(fx0 >= 0.0) || !(fy0 >= 0.0) || !(fx0 <= (double)(D.w - 2)) || !(fy0 <= (double)(D.h - 2))) return false;
  int ix = (int)fx0, iy = (int)fy0;
  double a = gx - fx0, b = gy - fy0;
  const float* p = D.d + (size_t)iy * D.w + ix;
  double d00 = __ldg(p), d10 = __ldg(p + 1), d01 = __ldg(p + D.w), d11 = __ldg(p + D.w + 1);
  z = (1 - b) * ((1 - a) * d00 + a * d10) + b * ((1 - a) * d01 + a * d11);
  zx = ((1 - b) * (d10 - d00) + b * (d11 - d01)) * D.ig;
  zy = ((1 - a) * (d01 - d00) + a * (d11 - d10)) * D.ig;
  return true;
}

__device__ __forceinline__ double height_above(const DsmView& D, const double* C, const double* w, double t) {
  double z, zx, zy;
  if (!dsm_sample(D, C[0] + t * w[0], C[1] + t * w[1], z, zx, zy)) return INFINITY;  // off the map = above
  return C[2] + t * w[2] - z;
}

// Range residual and 1x6 Jacobian at pose (R_cw, C). Warp-collective (all 32 lanes call it with the same
// arguments); the 64 march samples are evaluated 32 at a time, one per lane. Result is warp-uniform.
__device__ bool range_prior(const PassArgs& A, const double* R, const double* C, int lane, double& res, double (&J)[6]) {
  const DsmView D = make_dsm_view(A.dsm, A.dsm_w, A.dsm_h, A.dsm_ox, A.dsm_oy, A.dsm_gsd);
  double v[3] = {(double)A.ray[0], (double)A.ray[1], (double)A.ray[2]};
  double w[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = R[i] * v[0] + R[3 + i] * v[1] + R[6 + i] * v[2];   // R_cw^T v
  const double dm = (double)A.range_meas;
  double dist;
  if (A.prm.range_mode == PILOT_RANGE_HEIGHT) {
    dist = dm;
  } else {
    const int steps = A.prm.march_steps;
    const double dt = (double)A.prm.march_tfar_scale * dm / (double)steps;
    int found = -1;
    for (int i0 = 0; i0 < steps && found < 0; i0 += 32) {
      int i = i0 + lane;
      double f0 = height_above(D, C, w, (double)i * dt);
      double f1 = height_above(D, C, w, (double)(i + 1) * dt);
      unsigned hit = __ballot_sync(0xffffffffu, i < steps && f0 > 0.0 && f1 <= 0.0);
      if (hit) found = i0 + __ffs(hit) - 1;
    }
    if (found < 0) return false;
    double lo = (double)found * dt, hi = (double)(found + 1) * dt;
    for (int k = 0; k < A.prm.bisect_steps; ++k) {
      double mid = 0.5 * (lo + hi);
      if (height_above(D, C, w, mid) > 0.0) lo = mid; else hi = mid;
    }
    double flo = height_above(D, C, w, lo), fhi = height_above(D, C, w, hi);
    if (isfinite(flo) && isfinite(fhi) && flo - fhi > 0.0) dist = lo + (hi - lo) * flo * fast_rcp(flo - fhi);  // secant
    else dist = hi;
  }
  double z, zx, zy;
  double Pw[3] = {C[0] + dist * w[0], C[1] + dist * w[1], C[2] + dist * w[2]};           // Eq.(5)
  if (!dsm_sample(D, Pw[0], Pw[1], z, zx, zy)) return false;
  double n[3] = {-zx, -zy, 1.0};
  double ndw = 1.0;
  if (A.prm.range_mode == PILOT_RANGE_HEIGHT) {
    res = Pw[2] - z;                                                                     // Eq.(6)
  } else {
    res = dist - dm;
    ndw = n[0] * w[0] + n[1] * w[1] + n[2] * w[2];
    if (!(fabs(ndw) > 1e-12)) return false;
  }
  // row = n^T R_cw^T [ -I | [q]x ],  q = dist * v
  double m[3], q[3] = {dist * v[0], dist * v[1], dist * v[2]};
#pragma unroll
  for (int i = 0; i < 3; ++i) m[i] = R[3 * i] * n[0] + R[3 * i + 1] * n[1] + R[3 * i + 2] * n[2];
  J[0] = -m[0]; J[1] = -m[1]; J[2] = -m[2];
  J[3] = m[1] * q[2] - m[2] * q[1];      // (m^T [q]x)_0
  J[4] = m[2] * q[0] - m[0] * q[2];
  J[5] = m[0] * q[1] - m[1] * q[0];
  if (A.prm.range_mode == PILOT_RANGE_MARCH) {
    const double indw = fast_rcp(ndw);
#pragma unroll
    for (int i = 0; i < 6; ++i) J[i] = -J[i] * indw;
  }
  return true;
}

// ------------------------------------------------------------------ 6x6 Cholesky solve, SE(3) retraction (a9, a10)

// General path (any pivot): left-looking, returns false at the first pivot that is not positive and finite.
__device__ __noinline__ bool chol_solve6_checked(const double* Hs, double lambda, int damp_mode, const double* g, double* x) {
  double Lm[6][6], inv[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
#pragma unroll
    for (int j = 0; j <= i; ++j) {
      double s = Hs[tri(j, i)];
      if (i == j) s += (damp_mode == PILOT_DAMP_IDENTITY) ? lambda : lambda * fmax(Hs[tri(i, i)], 1e-12);
#pragma unroll
      for (int k = 0; k < j; ++k) s -= Lm[i][k] * Lm[j][k];
      if (i == j) {
        if (!(s > 0.0) || !isfinite(s)) return false;
        inv[i] = inv_sqrt(s);
        Lm[i][i] = s * inv[i];
      } else {
        Lm[i][j] = s * inv[j];
      }
    }
  }
  double y[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    double s = g[i];
#pragma unroll
    for (int k = 0; k < i; ++k) s -= Lm[i][k] * y[k];
    y[i] = s * inv[i];
  }
#pragma unroll
  for (int i = 5; i >= 0; --i) {
    double s = y[i];
#pragma unroll
    for (int k = 5; k > i; --k) s -= Lm[k][i] * x[k];
    x[i] = s * inv[i];
  }
  bool ok = true;
#pragma unroll
  for (int i = 0; i < 6; ++i) ok = ok && isfinite(x[i]);
  return ok;
}

// (H + damping) x = g by Cholesky. The finalisation is ONE lane's chain of dependent fp64 operations (8 cycles each on
// B200), so the common case is written for the shortest chain: right-looking (a column's updates of the trailing matrix
// are independent of each other: ~65 cycles per column = seed + cubic step + scale + update, against the left-looking
// accumulation whose chain grows with the column), no branch between the columns (one basic block for ptxas to
// interleave), substitutions column by column. Every element sees the same subtractions in the same order as in the
// left-looking form. A pivot outside (2^-1007, 2^993) - including every failure (<= 0, NaN, inf) - sends the whole solve
// to chol_solve6_checked on a cold path, which decides.
__device__ __forceinline__ bool chol_solve6(const double (&Hs)[21], double lambda, int damp_mode, const double (&g)[6], double (&x)[6],
                                            const double* H_mem, const double* g_mem /* the same system in memory, for the cold path */) {
  double a[21], inv[6];
#pragma unroll
  for (int i = 0; i < 21; ++i) a[i] = Hs[i];
#pragma unroll
  for (int i = 0; i < 6; ++i) a[tri(i, i)] += (damp_mode == PILOT_DAMP_IDENTITY) ? lambda : lambda * fmax(Hs[tri(i, i)], 1e-12);
  bool plain = true;
#pragma unroll
  for (int j = 0; j < 6; ++j) {
    const double d = a[tri(j, j)];
    plain = plain && d > 0.0 && fp64_mid_range(d);
    inv[j] = inv_sqrt_core(d);
#pragma unroll
    for (int i = j + 1; i < 6; ++i) a[tri(j, i)] *= inv[j];                 // L[i][j]
#pragma unroll
    for (int i = j + 1; i < 6; ++i)
#pragma unroll
      for (int k = j + 1; k <= i; ++k) a[tri(k, i)] -= a[tri(j, i)] * a[tri(j, k)];
  }
  double y[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) y[i] = g[i];
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    y[k] *= inv[k];
#pragma unroll
    for (int i = k + 1; i < 6; ++i) y[i] -= a[tri(k, i)] * y[k];
  }
#pragma unroll
  for (int k = 5; k >= 0; --k) {
    y[k] *= inv[k];
#pragma unroll
    for (int i = 0; i < k; ++i) y[i] -= a[tri(i, k)] * y[k];
  }
  bool ok = plain;
#pragma unroll
  for (int i = 0; i < 6; ++i) { x[i] = y[i]; ok = ok && isfinite(y[i]); }
  if (!plain) {                        // cold: works from memory so that the arrays above stay in registers
    double xs[6];
    const bool r = chol_solve6_checked(H_mem, lambda, damp_mode, g_mem, xs);
#pragma unroll
    for (int i = 0; i < 6; ++i) x[i] = xs[i];
    return r;
  }
  return ok;
}

// sin(th)/th, (1 - cos th)/th^2, (th - sin th)/th^3 as even power series in th, TERMS terms each (three independent
// Horner chains)
template <int TERMS>
__device__ __forceinline__ void so3_series(double th2, double& a, double& b, double& c) {
  constexpr double f[22] = {1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320,
                            1.0 / 362880, 1.0 / 3628800, 1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0,
                            1.0 / 87178291200.0, 1.0 / 1307674368000.0, 1.0 / 20922789888000.0,
                            1.0 / 355687428096000.0, 1.0 / 6402373705728000.0, 1.0 / 121645100408832000.0,
                            1.0 / 2432902008176640000.0, 1.0 / 51090942171709440000.0};
  a = f[2 * TERMS - 1]; b = f[2 * TERMS]; c = f[2 * TERMS + 1];
#pragma unroll
  for (int k = TERMS - 2; k >= 0; --k) {
    a = f[2 * k + 1] - th2 * a;
    b = f[2 * k + 2] - th2 * b;
    c = f[2 * k + 3] - th2 * c;
  }
}

// T_cw <- exp(xi) T_cw (Eq.9): R' = E R, C' = C - R^T E^T V rho with E = exp([phi]x) = I + a K + b K^2, V = I + b K + c K^2,
// K^2 = phi phi^T - th^2 I, and E^T V = V(-phi) (E^T V(phi) = int_0^1 exp((t-1) K) dt), so that
// E^T V rho = rho - b (phi x rho) + c (phi x (phi x rho)). Written for few instructions: one lane runs it as a dependent chain.
__device__ __forceinline__ void retract(const double* R, const double* C, const double (&xi)[6], double* Rn, double* Cn) {
  const double px = xi[3], py = xi[4], pz = xi[5];
  const double th2 = px * px + py * py + pz * pz;
  double a, b, c;
  if (th2 <= 1e-2) {
    so3_series<5>(th2, a, b, c);         // LM steps are small rotations: next term < 3e-18 at th = 0.1
  } else if (th2 <= 0.25) {
    so3_series<10>(th2, a, b, c);        // next term < 3e-23 at th = 0.5
  } else {
    const double th = sqrt(th2);
    double sn, cs;
    sincos(th, &sn, &cs);
    a = sn / th; b = (1.0 - cs) / th2; c = (th - sn) / (th2 * th);
  }
  // E: diagonal 1 + b (p_i^2 - th2), off-diagonal b p_i p_j -+ a p_k
  const double bxy = b * (px * py), bxz = b * (px * pz), byz = b * (py * pz);
  const double E[9] = {fma(b, px * px - th2, 1.0), fma(-a, pz, bxy), fma(a, py, bxz),
                       fma(a, pz, bxy), fma(b, py * py - th2, 1.0), fma(-a, px, byz),
                       fma(-a, py, bxz), fma(a, px, byz), fma(b, pz * pz - th2, 1.0)};
  // w = E^T V rho = rho - b k1 + c k2, k1 = phi x rho, k2 = phi x k1
  const double k1x = py * xi[2] - pz * xi[1], k1y = pz * xi[0] - px * xi[2], k1z = px * xi[1] - py * xi[0];
  const double k2x = py * k1z - pz * k1y, k2y = pz * k1x - px * k1z, k2z = px * k1y - py * k1x;
  const double wx = fma(c, k2x, fma(-b, k1x, xi[0])), wy = fma(c, k2y, fma(-b, k1y, xi[1])), wz = fma(c, k2z, fma(-b, k1z, xi[2]));
  double Rt[9];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) Rt[3 * i + j] = E[3 * i] * R[j] + E[3 * i + 1] * R[3 + j] + E[3 * i + 2] * R[6 + j];
#pragma unroll
  for (int i = 0; i < 3; ++i) Cn[i] = C[i] - (R[i] * wx + R[3 + i] * wy + R[6 + i] * wz);
#pragma unroll
  for (int i = 0; i < 9; ++i) Rn[i] = Rt[i];
}

}  // namespace

namespace {

// ------------------------------------------------------------------ per-hypothesis finalisation (a6-a11), one warp

__device__ void write_final(const PassArgs& A, const HypState& s, int m) {
  if (A.out.poses_dev) {
    float* T = A.out.poses_dev + 12 * (size_t)m;
    for (int i = 0; i < 3; ++i) {
      for (int k = 0; k < 3; ++k) T[4 * i + k] = (float)s.R[3 * k + i];     // R_wc = R_cw^T
      T[4 * i + 3] = (float)s.C[i];
    }
  }
  if (A.out.cost_dev) A.out.cost_dev[m] = (float)s.cost;
  if (A.out.n_valid_dev) A.out.n_valid_dev[m] = s.n_valid;
  if (A.out.status_dev) A.out.status_dev[m] = s.status | s.flags;
}

// What the two priors add to the photo sums at a candidate pose (supp Eq.5-6): they depend on the pose only, so the resident
// kernel evaluates them on a warp of their own WHILE the others gather, and the finalisation just adds 28 numbers.
struct PriorTerms { double H[21]; double g[6]; double cost; unsigned flags; };

__device__ __forceinline__ bool range_enabled(const PassArgs& A) {
  return A.prm.range_mode != PILOT_RANGE_OFF && A.prm.w_range > 0.f && A.dsm != nullptr;
}

// Warp-collective (the ray-march runs on the whole warp); lane 0 returns the terms in registers.
__device__ __forceinline__ void prior_terms(const PassArgs& A, const double* Rc, const double* Cc, int lane, double (&Hp)[21],
                                            double (&gp)[6], double& costp, unsigned& fl) {
  const pilot_refine_params& P = A.prm;
  double rr = 0.0, Jr[6];
  const bool range_on = range_enabled(A);
  bool range_ok = false;
  if (range_on) range_ok = range_prior(A, Rc, Cc, lane, rr, Jr);
#pragma unroll
  for (int i = 0; i < 21; ++i) Hp[i] = 0.0;
#pragma unroll
  for (int i = 0; i < 6; ++i) gp[i] = 0.0;
  costp = 0.0; fl = 0u;
  if (lane != 0) return;
  if (P.w_gravity > 0.f) {                                                   // Eq.(3)
    double e[3], r[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      e[i] = Rc[3 * i] * A.pd.gw[0] + Rc[3 * i + 1] * A.pd.gw[1] + Rc[3 * i + 2] * A.pd.gw[2];
      r[i] = e[i] - A.pd.gi[i];
    }
    double rho, drho;
    robust_d(P.loss, r[0] * r[0] + r[1] * r[1] + r[2] * r[2], A.pd.gravity_scale, rho, drho);
    const double wg = A.pd.w_gravity * drho;
    // J = [0 | -[e]x]: J^T r = e x r, J^T J = |e|^2 I - e e^T
    const double ee = e[0] * e[0] + e[1] * e[1] + e[2] * e[2];
    gp[3] = wg * (e[1] * r[2] - e[2] * r[1]);
    gp[4] = wg * (e[2] * r[0] - e[0] * r[2]);
    gp[5] = wg * (e[0] * r[1] - e[1] * r[0]);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) Hp[tri(3 + a, 3 + b)] = wg * ((a == b ? ee : 0.0) - e[a] * e[b]);
    costp = A.pd.w_gravity * rho;
  }
  if (range_on) {                                                            // Eq.(5)-(6) / ray-march
    if (range_ok) {
      double rho, drho;
      robust_d(P.loss, rr * rr, A.pd.range_scale, rho, drho);
      const double wr = A.pd.w_range * drho;
#pragma unroll
      for (int a = 0; a < 6; ++a) {
        const double wj = wr * Jr[a];
        gp[a] += wj * rr;
#pragma unroll
        for (int b = a; b < 6; ++b) Hp[tri(a, b)] += wj * Jr[b];
      }
      costp += A.pd.w_range * rho;
    } else {
      fl |= PILOT_STATUS_RANGE_SKIP;
    }
  }
}

// The same into memory (shared): what the resident kernel's prior warp calls.
__device__ __forceinline__ void prior_terms_store(const PassArgs& A, const double* Rc, const double* Cc, int lane, PriorTerms* out) {
  double Hp[21], gp[6], costp;
  unsigned fl;
  prior_terms(A, Rc, Cc, lane, Hp, gp, costp, fl);
  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < 21; ++i) out->H[i] = Hp[i];
#pragma unroll
    for (int i = 0; i < 6; ++i) out->g[i] = gp[i];
    out->cost = costp; out->flags = fl;
  }
}

// Lane 0 does everything after the warp-wide ray-march; what it runs is ONE chain of dependent fp64 operations (8 cycles
// each on B200, and a DFMA occupies the issue slot for 2), so the code is written for few instructions and a short chain:
// the accepted system goes to the solve in registers (not through the state), the priors arrive as 28 numbers to add.
// A lane-parallel variant (component i of the system in lane i, the record stores and state copies spread over the lanes,
// a 6x6 Cholesky by rows with shuffle broadcasts) was written in round 2, parity green, and removed: 8.3 k cycles per
// iteration against 6.7 k for the serial one of that time (3.1 k after the rewrite above; 2.x k now) - shuffles and
// selects only lengthen the chain.
// Warp-collective. `s` is the hypothesis' optimiser state (shared memory); `sums` the photo sums in double (shared memory);
// `pre` = the priors' terms at the candidate pose if they were computed already, else nullptr (computed here).
__device__ void finalize_hypothesis(const PassArgs& A, HypState& s, int m, const double* sums /* smem, kNacc */, int lane,
                                    const PriorTerms* pre) {
  const pilot_refine_params& P = A.prm;

  double Hn[21], gn[6], costn;
  unsigned fl = 0;
  if (pre) {
    if (lane != 0) return;
#pragma unroll
    for (int i = 0; i < 21; ++i) Hn[i] = pre->H[i];
#pragma unroll
    for (int i = 0; i < 6; ++i) gn[i] = pre->g[i];
    costn = pre->cost; fl = pre->flags;
  } else {
    prior_terms(A, s.Rc, s.Cc, lane, Hn, gn, costn, fl);
    if (lane != 0) return;
  }
#ifdef PILOT_FIN_PROFILE
  long long tp[6]; tp[0] = clock64();
#define PILOT_TP(i) tp[i] = clock64();
#else
#define PILOT_TP(i)
#endif
#pragma unroll
  for (int i = 0; i < 21; ++i) Hn[i] += sums[i];          // converted to double by the 32 lanes that summed them
#pragma unroll
  for (int i = 0; i < 6; ++i) gn[i] += sums[21 + i];
  costn += sums[27];
  const int nv = (int)(sums[28] + 0.5);
  s.visible_evals += (unsigned long long)nv;
  if (nv < P.min_valid) { costn = INFINITY; fl |= PILOT_STATUS_FEW_VALID; }
  if (isnan(costn)) s.status |= PILOT_STATUS_NONFINITE;
  PILOT_TP(1)

  // accept / reject (a10). The first evaluation of a level is taken unconditionally.
  double lam = s.lambda;
  const bool first = s.pending == 0;
  if (first || P.lm_mode == PILOT_LM_FIXED || costn < s.cost) {
#pragma unroll
    for (int i = 0; i < 9; ++i) s.R[i] = s.Rc[i];
#pragma unroll
    for (int i = 0; i < 3; ++i) s.C[i] = s.Cc[i];
#pragma unroll
    for (int i = 0; i < 21; ++i) s.H[i] = Hn[i];
#pragma unroll
    for (int i = 0; i < 6; ++i) s.g[i] = gn[i];
    s.cost = costn; s.n_valid = nv; s.flags = fl;
    if (!first && P.lm_mode == PILOT_LM_ADAPTIVE) lam = fmax(lam * A.pd.lambda_down, A.pd.lambda_min);
    if (!first && A.iter_accept) A.iter_accept[(size_t)(A.rec_base + s.k - 1) * (size_t)A.n_hyp + (size_t)m] = 1;   // the step of record k - 1
  } else {                                                                   // the accepted state stays: the solve reads it back
#pragma unroll
    for (int i = 0; i < 21; ++i) Hn[i] = s.H[i];
#pragma unroll
    for (int i = 0; i < 6; ++i) gn[i] = s.g[i];
    costn = s.cost;
    lam = fmin(lam * A.pd.lambda_up, A.pd.lambda_max);
  }
  // from here on (Hn, gn, costn) = the ACCEPTED system, in registers for the first solve

  PILOT_TP(2)
  // record + damped solve (a9, Eq.8); a failed factorisation consumes the iteration and raises lambda
  bool have = false;
  const size_t Hn_ = (size_t)A.n_hyp;
  int k = s.k;
  bool again = false;
  while (k < A.iters) {
    if (again) {                                                             // cold: registers were given up after the first try
#pragma unroll
      for (int i = 0; i < 21; ++i) Hn[i] = s.H[i];
#pragma unroll
      for (int i = 0; i < 6; ++i) gn[i] = s.g[i];
    }
    again = true;
    const size_t ri = (size_t)(A.rec_base + k) * Hn_ + (size_t)m;
    if (A.out.iter_hessian_dev) {
      float* o = A.out.iter_hessian_dev + 36 * ri;
#pragma unroll
      for (int a = 0; a < 6; ++a)
#pragma unroll
        for (int b = a; b < 6; ++b) { const float v = (float)Hn[tri(a, b)]; o[6 * a + b] = v; if (b != a) o[6 * b + a] = v; }
    }
    if (A.out.iter_gradient_dev)
#pragma unroll
      for (int a = 0; a < 6; ++a) A.out.iter_gradient_dev[6 * ri + a] = (float)gn[a];
    if (A.out.iter_cost_dev) A.out.iter_cost_dev[ri] = (float)costn;
    if (A.out.iter_lambda_dev) A.out.iter_lambda_dev[ri] = (float)lam;
    if (A.iter_accept) A.iter_accept[ri] = 0;                                // set when (if) this record's step is accepted
    if (A.iter_poses) {
      float* T = A.iter_poses + 12 * ri;
      for (int i = 0; i < 3; ++i) {
        for (int c = 0; c < 3; ++c) T[4 * i + c] = (float)s.R[3 * c + i];    // R_wc = R_cw^T
        T[4 * i + 3] = (float)s.C[i];
      }
    }
    double dxi[6];
    PILOT_TP(3)
    const bool ok = chol_solve6(Hn, lam, P.damp_mode, gn, dxi, s.H, s.g);
    PILOT_TP(4)
    k += 1;
    if (ok) {
#pragma unroll
      for (int i = 0; i < 6; ++i) dxi[i] = -dxi[i];
      retract(s.R, s.C, dxi, s.Rc, s.Cc);                                    // Eq.(9)
      PILOT_TP(5)
      s.pending = 1;
      have = true;
      break;
    }
    if (lam >= A.pd.lambda_max) s.status |= PILOT_STATUS_CHOL_FAIL;
    lam = fmin(lam * A.pd.lambda_up, A.pd.lambda_max);
  }
  s.k = k;
  s.lambda = lam;
  if (!have) {                                                               // this level is finished
    s.level = A.level + 1;
    s.k = 0; s.pending = 0; s.lambda = A.pd.lambda_init;
#pragma unroll
    for (int i = 0; i < 9; ++i) s.Rc[i] = s.R[i];
#pragma unroll
    for (int i = 0; i < 3; ++i) s.Cc[i] = s.C[i];
    if (A.level + 1 == A.level_end) write_final(A, s, m);
  }
#ifdef PILOT_FIN_PROFILE
  if (have) { float* o = A.partials + (size_t)m * 32 + 24; for (int i = 0; i < 5; ++i) o[i] += (float)(tp[i + 1] - tp[i]); o[5] += 1.f; }
#endif
#undef PILOT_TP
}

// The same on the state in the workspace (global memory): the warp stages it through `scratch` (SHARED memory, one
// HypState per calling warp) with coalesced copies, so that lane 0 works on shared memory instead of chasing 456 bytes
// of global memory through dependent loads (config 4 7.75 -> 7.57 ms, config 2 7.41 -> 7.33). Warp-collective.
__device__ __noinline__ void finalize_in_workspace(const PassArgs& A, int m, const double* sums, int lane, HypState* scratch,
                                                   const PriorTerms* pre = nullptr) {
  const int* src = reinterpret_cast<const int*>(A.state + m);
  int* dst = reinterpret_cast<int*>(scratch);
  for (int i = lane; i < (int)(sizeof(HypState) / 4); i += 32) dst[i] = src[i];
  __syncwarp();
  finalize_hypothesis(A, *scratch, m, sums, lane, pre);
  __syncwarp();
  int* out = reinterpret_cast<int*>(A.state + m);
  for (int i = lane; i < (int)(sizeof(HypState) / 4); i += 32) out[i] = dst[i];
}

}  // namespace
