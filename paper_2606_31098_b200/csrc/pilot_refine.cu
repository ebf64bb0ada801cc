// pilot_refine.cu — B200 (sm_100a) implementation of include/pilot_refine.h.
//
// One launch per EVAL pass: the photo kernel projects every
// (anchor, hypothesis) unit, gathers the 2x2 bilinear footprint of the query feature map with
// 16-byte channel-vector loads coalesced along C, forms the per-unit 2x2 Gram / residual
// scalars, lifts them through the 2x6 projection Jacobian and reduces them per hypothesis.
// The last CTA to finish a hypothesis reduces the per-chunk partials in a fixed order
// (deterministic), adds the gravity and range priors (heightfield ray-march), takes the LM
// accept/reject decision, solves the damped 6x6 system, retracts on SE(3) and publishes the
// candidate pose for the next pass — no host synchronisation anywhere.
//
// Shares no code with oracle/ (only the POD structs of include/pilot_refine.h).
#include "../../include/pilot_refine.h"

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

namespace {

constexpr int kThreads = 256;            // threads per CTA of the photo kernel
constexpr int kWarps = kThreads / 32;
constexpr int kNacc = 32;                // 21 H + 6 g + cost + n_valid, padded to 32 floats
constexpr int kMinChunk = kWarps * 32;   // one 32-unit batch per warp

// index of the upper-triangular entry (a<=b) in the packed 21-vector
__host__ __device__ constexpr int tri(int a, int b) { return a * 6 - a * (a - 1) / 2 + (b - a); }

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
  HypState* state;
  float* partials;          // [n_hyp][n_chunks][kNacc]
  unsigned* counters;       // [n_hyp]
  pilot_refine_outputs out;
};

// ------------------------------------------------------------------ element decoding

struct F32Tag { static constexpr int kVec = 4; };
struct BF16Tag { static constexpr int kVec = 8; };
struct F16Tag { static constexpr int kVec = 8; };

__device__ __forceinline__ uint4 ldg16(const void* p) {
  return __ldg(reinterpret_cast<const uint4*>(p));
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

// ------------------------------------------------------------------ the photo kernel
//
// grid = (n_hyp, n_chunks): blockIdx.x (fastest) is the hypothesis, so CTAs that run together
// sweep the SAME chunk of (spatially sorted) anchors under different poses and the union of their
// footprints is a narrow band of the map that stays in L2.
template <class T, int G, bool CEN>
__global__ void __launch_bounds__(kThreads) photo_pass_kernel(const __grid_constant__ PassArgs A);

template <class T, int G, bool CEN>
__device__ __forceinline__ void photo_accumulate(const PassArgs& A, const HypState* st, int chunk_idx,
                                                 float (&acc)[kNacc]) {
  constexpr int LOG = Log2<G>::v;
  const LevelArgs& L = A.lv;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int sub = lane & (G - 1);
  const unsigned esz = 16 / T::kVec;
  const unsigned px_stride = (unsigned)L.C * esz;
  const unsigned row_stride = px_stride * (unsigned)L.W;
  const char* feat = static_cast<const char*>(L.feat);
  const char* refb = static_cast<const char*>(L.ref);

  // candidate pose (the pose this pass evaluates), double for the projection
  double R[9], Cc[3];
#pragma unroll
  for (int i = 0; i < 9; ++i) R[i] = st->Rc[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) Cc[i] = st->Cc[i];

  const int begin = chunk_idx * A.chunk;
  const int end = min(begin + A.chunk, L.N);
  const float wmax = (float)(L.W - 1), hmax = (float)(L.H - 1);

  for (int base = begin + warp * 32; base < end; base += kWarps * 32) {
    // ---- lane-per-unit: projection + visibility (a2), in double so that u,v carry no fp32 noise
    const int j = base + lane;
    bool valid = j < end;
    float4 P = valid ? __ldg(L.points + j) : make_float4(0.f, 0.f, 0.f, 0.f);
    double dx = (double)P.x - Cc[0], dy = (double)P.y - Cc[1], dz = (double)P.z - Cc[2];
    double Xd = R[0] * dx + R[1] * dy + R[2] * dz;
    double Yd = R[3] * dx + R[4] * dy + R[5] * dz;
    double Zd = R[6] * dx + R[7] * dy + R[8] * dz;
    valid = valid && (Zd > (double)A.prm.z_near);
    double izd = 1.0 / Zd;
    double ud = (double)L.fx * Xd * izd + (double)L.cx;
    double vd = (double)L.fy * Yd * izd + (double)L.cy;
    double x0d = floor(ud), y0d = floor(vd);
    valid = valid && (x0d >= 0.0) && (y0d >= 0.0) && (x0d + 1.0 <= (double)wmax) && (y0d + 1.0 <= (double)hmax);
    float a = valid ? (float)(ud - x0d) : 0.f;
    float b = valid ? (float)(vd - y0d) : 0.f;
    int x0 = valid ? (int)x0d : 0, y0 = valid ? (int)y0d : 0;
    unsigned off = ((unsigned)y0 * (unsigned)L.W + (unsigned)x0) * px_stride;   // invalid units read pixel (0,0)
    unsigned offv = valid ? off : 0xffffffffu;

    // ---- group rounds: gather + per-unit contraction (a3-a5), reduce-scatter so that lane i ends
    //      up with the six sums of unit i of this batch
    float stash[LOG > 0 ? LOG : 1][6];
    float cur[6];
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
    float na, nb; bool nvalid;
    RawTaps nxt;
    unsigned cflags = 0;                                   // CEN: which outer taps are clamped at the border
    if constexpr (CEN) cflags = (x0 > 0 ? 1u : 0u) | (x0 + 2 <= L.W - 1 ? 2u : 0u) | (y0 > 0 ? 4u : 0u) | (y0 + 2 <= L.H - 1 ? 8u : 0u);
    else nxt = fetch(0, na, nb, nvalid);
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
        RawTaps t = nxt;
        float ra = na, rb = nb;
        rvalid = nvalid;
        if (r + 1 < G) nxt = fetch(r + 1, na, nb, nvalid);   // software pipeline: next unit's loads in flight
        unit_partials<T>(t, ra, rb, cur);
      }
      if (!rvalid) {
#pragma unroll
        for (int i = 0; i < 6; ++i) cur[i] = 0.f;
      }
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
        for (int q = p; q < 6; ++q) acc[tri(p, q)] += mu * Ju[q] + mv * Jv[q];
        acc[21 + p] += b1 * Ju[p] + b2 * Jv[p];
      }
      acc[27] += rho;
      acc[28] += 1.f;
    }
  }
}

}  // namespace

namespace {

// ------------------------------------------------------------------ priors (a7, a8), executed by one full warp in double

struct DsmView { const float* d; int w, h; double ox, oy, gsd; };

// Bilinear heightfield sample and exact gradient (per metre). false = outside the DSM.
__device__ __forceinline__ bool dsm_sample(const DsmView& D, double x, double y, double& z, double& zx, double& zy) {
  double gx = (x - D.ox) / D.gsd, gy = (y - D.oy) / D.gsd;
  double fx0 = floor(gx), fy0 = floor(gy);
  if (!(fx0 >= 0.0) || !(fy0 >= 0.0) || !(fx0 <= (double)(D.w - 2)) || !(fy0 <= (double)(D.h - 2))) return false;
  int ix = (int)fx0, iy = (int)fy0;
  double a = gx - fx0, b = gy - fy0;
  const float* p = D.d + (size_t)iy * D.w + ix;
  double d00 = __ldg(p), d10 = __ldg(p + 1), d01 = __ldg(p + D.w), d11 = __ldg(p + D.w + 1);
  z = (1 - b) * ((1 - a) * d00 + a * d10) + b * ((1 - a) * d01 + a * d11);
  zx = ((1 - b) * (d10 - d00) + b * (d11 - d01)) / D.gsd;
  zy = ((1 - a) * (d01 - d00) + a * (d11 - d10)) / D.gsd;
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
  DsmView D{A.dsm, A.dsm_w, A.dsm_h, (double)A.dsm_ox, (double)A.dsm_oy, (double)A.dsm_gsd};
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
    if (isfinite(flo) && isfinite(fhi) && flo - fhi > 0.0) dist = lo + (hi - lo) * flo / (flo - fhi);  // secant
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
#pragma unroll
    for (int i = 0; i < 6; ++i) J[i] = -J[i] / ndw;
  }
  return true;
}

// ------------------------------------------------------------------ 6x6 Cholesky solve, SE(3) retraction (a9, a10)

__device__ bool chol_solve6(const double (&Hs)[21], double lambda, int damp_mode, const double (&g)[6], double (&x)[6]) {
  double Lm[6][6];
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
        Lm[i][i] = sqrt(s);
      } else {
        Lm[i][j] = s / Lm[j][j];
      }
    }
  }
  double y[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    double s = g[i];
#pragma unroll
    for (int k = 0; k < i; ++k) s -= Lm[i][k] * y[k];
    y[i] = s / Lm[i][i];
  }
#pragma unroll
  for (int i = 5; i >= 0; --i) {
    double s = y[i];
#pragma unroll
    for (int k = i + 1; k < 6; ++k) s -= Lm[k][i] * x[k];
    x[i] = s / Lm[i][i];
  }
  bool ok = true;
#pragma unroll
  for (int i = 0; i < 6; ++i) ok = ok && isfinite(x[i]);
  return ok;
}

// T_cw <- exp(xi) T_cw (Eq.9): R' = E R, C' = C - R^T E^T V rho
__device__ void retract(const double* R, const double* C, const double (&xi)[6], double* Rn, double* Cn) {
  const double px = xi[3], py = xi[4], pz = xi[5];
  double th2 = px * px + py * py + pz * pz, th = sqrt(th2);
  double a, b, c;
  if (th < 1e-4) {
    a = 1.0 - th2 / 6.0 + th2 * th2 / 120.0;
    b = 0.5 - th2 / 24.0 + th2 * th2 / 720.0;
    c = 1.0 / 6.0 - th2 / 120.0 + th2 * th2 / 5040.0;
  } else {
    a = sin(th) / th; b = (1.0 - cos(th)) / th2; c = (th - sin(th)) / (th2 * th);
  }
  double K[9] = {0, -pz, py, pz, 0, -px, -py, px, 0}, K2[9], E[9], V[9];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) K2[3 * i + j] = K[3 * i] * K[j] + K[3 * i + 1] * K[3 + j] + K[3 * i + 2] * K[6 + j];
  for (int i = 0; i < 9; ++i) {
    double I = (i % 4 == 0) ? 1.0 : 0.0;
    E[i] = I + a * K[i] + b * K2[i];
    V[i] = I + b * K[i] + c * K2[i];
  }
  double Vr[3], EtVr[3], Rt[9];
  for (int i = 0; i < 3; ++i) Vr[i] = V[3 * i] * xi[0] + V[3 * i + 1] * xi[1] + V[3 * i + 2] * xi[2];
  for (int i = 0; i < 3; ++i) EtVr[i] = E[i] * Vr[0] + E[3 + i] * Vr[1] + E[6 + i] * Vr[2];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) Rt[3 * i + j] = E[3 * i] * R[j] + E[3 * i + 1] * R[3 + j] + E[3 * i + 2] * R[6 + j];
  for (int i = 0; i < 3; ++i) Cn[i] = C[i] - (R[i] * EtVr[0] + R[3 + i] * EtVr[1] + R[6 + i] * EtVr[2]);
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

__device__ void finalize_hypothesis(const PassArgs& A, int m, const float* sums /* smem, kNacc */, int lane) {
  HypState& s = A.state[m];
  const pilot_refine_params& P = A.prm;

  // range prior at the evaluated pose: warp-collective
  double rr = 0.0, Jr[6];
  bool range_on = P.range_mode != PILOT_RANGE_OFF && P.w_range > 0.f && A.dsm != nullptr;
  bool range_ok = false;
  if (range_on) range_ok = range_prior(A, s.Rc, s.Cc, lane, rr, Jr);
  if (lane != 0) return;

  double Hn[21], gn[6], costn;
  unsigned fl = 0;
  for (int i = 0; i < 21; ++i) Hn[i] = (double)sums[i];
  for (int i = 0; i < 6; ++i) gn[i] = (double)sums[21 + i];
  costn = (double)sums[27];
  int nv = (int)(sums[28] + 0.5f);
  if (nv < P.min_valid) { costn = INFINITY; fl |= PILOT_STATUS_FEW_VALID; }

  if (P.w_gravity > 0.f) {                                                   // Eq.(3)
    double e[3], r[3];
    for (int i = 0; i < 3; ++i) {
      e[i] = s.Rc[3 * i] * (double)A.gw[0] + s.Rc[3 * i + 1] * (double)A.gw[1] + s.Rc[3 * i + 2] * (double)A.gw[2];
      r[i] = e[i] - (double)A.gi[i];
    }
    double rho, drho;
    robust<double>(P.loss, r[0] * r[0] + r[1] * r[1] + r[2] * r[2], (double)P.gravity_scale, rho, drho);
    double wg = (double)P.w_gravity * drho;
    // J = [0 | -[e]x]; rows of -[e]x: (0, e2, -e1), (-e2, 0, e0), (e1, -e0, 0)
    double Jg[3][3] = {{0, e[2], -e[1]}, {-e[2], 0, e[0]}, {e[1], -e[0], 0}};
    for (int a = 0; a < 3; ++a) {
      double ga = 0;
      for (int i = 0; i < 3; ++i) ga += Jg[i][a] * r[i];
      gn[3 + a] += wg * ga;
      for (int b = a; b < 3; ++b) {
        double h = 0;
        for (int i = 0; i < 3; ++i) h += Jg[i][a] * Jg[i][b];
        Hn[tri(3 + a, 3 + b)] += wg * h;
      }
    }
    costn += (double)P.w_gravity * rho;
  }
  if (range_on) {                                                            // Eq.(5)-(6) / ray-march
    if (range_ok) {
      double rho, drho;
      robust<double>(P.loss, rr * rr, (double)P.range_scale, rho, drho);
      double wr = (double)P.w_range * drho;
      for (int a = 0; a < 6; ++a) {
        gn[a] += wr * Jr[a] * rr;
        for (int b = a; b < 6; ++b) Hn[tri(a, b)] += wr * Jr[a] * Jr[b];
      }
      costn += (double)P.w_range * rho;
    } else {
      fl |= PILOT_STATUS_RANGE_SKIP;
    }
  }
  if (isnan(costn)) s.status |= PILOT_STATUS_NONFINITE;

  // accept / reject (a10). The first evaluation of a level is taken unconditionally.
  double lam = s.lambda;
  const bool first = s.pending == 0;
  if (first || P.lm_mode == PILOT_LM_FIXED || costn < s.cost) {
    for (int i = 0; i < 9; ++i) s.R[i] = s.Rc[i];
    for (int i = 0; i < 3; ++i) s.C[i] = s.Cc[i];
    for (int i = 0; i < 21; ++i) s.H[i] = Hn[i];
    for (int i = 0; i < 6; ++i) s.g[i] = gn[i];
    s.cost = costn; s.n_valid = nv; s.flags = fl;
    if (!first && P.lm_mode == PILOT_LM_ADAPTIVE) lam = fmax(lam * (double)P.lambda_down, (double)P.lambda_min);
  } else {
    lam = fmin(lam * (double)P.lambda_up, (double)P.lambda_max);
  }

  // record + damped solve (a9, Eq.8); a failed factorisation consumes the iteration and raises lambda
  bool have = false;
  const size_t Hn_ = (size_t)A.n_hyp;
  while (s.k < A.iters) {
    const size_t ri = (size_t)(A.rec_base + s.k) * Hn_ + (size_t)m;
    if (A.out.iter_hessian_dev) {
      float* o = A.out.iter_hessian_dev + 36 * ri;
      for (int a = 0; a < 6; ++a)
        for (int b = 0; b < 6; ++b) o[6 * a + b] = (float)s.H[a <= b ? tri(a, b) : tri(b, a)];
    }
    if (A.out.iter_gradient_dev) for (int a = 0; a < 6; ++a) A.out.iter_gradient_dev[6 * ri + a] = (float)s.g[a];
    if (A.out.iter_cost_dev) A.out.iter_cost_dev[ri] = (float)s.cost;
    if (A.out.iter_lambda_dev) A.out.iter_lambda_dev[ri] = (float)lam;
    double dxi[6];
    bool ok = chol_solve6(s.H, lam, P.damp_mode, s.g, dxi);
    s.k += 1;
    if (ok) {
      for (int i = 0; i < 6; ++i) dxi[i] = -dxi[i];
      retract(s.R, s.C, dxi, s.Rc, s.Cc);                                    // Eq.(9)
      s.pending = 1;
      have = true;
      break;
    }
    if (lam >= (double)P.lambda_max) s.status |= PILOT_STATUS_CHOL_FAIL;
    lam = fmin(lam * (double)P.lambda_up, (double)P.lambda_max);
  }
  s.lambda = lam;
  if (!have) {                                                               // this level is finished
    s.level = A.level + 1;
    s.k = 0; s.pending = 0; s.lambda = (double)P.lambda_init;
    for (int i = 0; i < 9; ++i) s.Rc[i] = s.R[i];
    for (int i = 0; i < 3; ++i) s.Cc[i] = s.C[i];
    if (A.level + 1 == A.level_end) write_final(A, s, m);
  }
}

// ------------------------------------------------------------------ kernels

template <class T, int G, bool CEN>
__global__ void __launch_bounds__(kThreads) photo_pass_kernel(const __grid_constant__ PassArgs A) {
  const int m = blockIdx.x, chunk_idx = blockIdx.y;
  const HypState* st = A.state + m;
  if (st->level != A.level) return;             // finished this level early (failed factorisations)

  float acc[kNacc];
#pragma unroll
  for (int i = 0; i < kNacc; ++i) acc[i] = 0.f;
  photo_accumulate<T, G, CEN>(A, st, chunk_idx, acc);

  // reduce-scatter over the warp: lane i ends with the warp total of component i (31 shuffles)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
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
  __shared__ float s_part[kWarps][kNacc];
  __shared__ float s_sum[kNacc];
  __shared__ int s_last;
  s_part[warp][lane] = acc[0];
  __syncthreads();
  if (warp == 0) {
    float t = 0.f;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) t += s_part[w][lane];                    // fixed order
    A.partials[((size_t)m * A.n_chunks + chunk_idx) * kNacc + lane] = t;
    __threadfence();
    __syncwarp();
    if (lane == 0) s_last = (atomicAdd(A.counters + m, 1u) == (unsigned)(A.n_chunks - 1));
  }
  __syncthreads();
  if (!s_last || warp != 0) return;

  // last CTA of this hypothesis: fixed-order sum over chunks (deterministic), then the LM step
  __threadfence();
  float t = 0.f;
  const float* p = A.partials + (size_t)m * A.n_chunks * kNacc + lane;
  for (int c = 0; c < A.n_chunks; ++c) t += __ldcg(p + (size_t)c * kNacc);
  s_sum[lane] = t;
  if (lane == 0) A.counters[m] = 0u;
  __syncwarp();
  finalize_hypothesis(A, m, s_sum, lane);
}

__global__ void init_state_kernel(HypState* state, unsigned* counters, const float* poses, int n_hyp, double lambda_init,
                                  int level_begin) {
  int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n_hyp) return;
  HypState s;
  const float* T = poses + 12 * (size_t)m;
  for (int i = 0; i < 3; ++i) {
    for (int k = 0; k < 3; ++k) s.R[3 * k + i] = (double)T[4 * i + k];       // R_cw = R_wc^T
    s.C[i] = (double)T[4 * i + 3];
  }
  for (int i = 0; i < 9; ++i) s.Rc[i] = s.R[i];
  for (int i = 0; i < 3; ++i) s.Cc[i] = s.C[i];
  for (int i = 0; i < 21; ++i) s.H[i] = 0.0;
  for (int i = 0; i < 6; ++i) s.g[i] = 0.0;
  s.cost = 0.0; s.lambda = lambda_init; s.n_valid = 0; s.flags = 0; s.status = 0;
  s.level = level_begin; s.k = 0; s.pending = 0;
  state[m] = s;
  counters[m] = 0u;
}

}  // namespace

// ====================================================================== host side

struct pilot_refine_handle {
  pilot_refine_config cfg;
  char* ws;                 // device scratch
  size_t ws_bytes;
  bool owns_ws;
  int max_chunks;
  int chunk_override;       // 0 = heuristic
  int sm_count;
  int last_launches;
  // host-path staging (create_host only)
  bool host_mode;
  int max_dsm_w, max_dsm_h;
  char* stage;              // one cudaMalloc
  size_t stage_bytes;
};

namespace {

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
size_t elem_size(pilot_dtype d) { return d == PILOT_F32 ? 4 : 2; }

// lanes per unit: C*sizeof/16, must be a power of two in [1, 32]
int lanes_per_unit(int channels, pilot_dtype d) {
  size_t bytes = (size_t)channels * elem_size(d);
  if (channels <= 0 || bytes % 16 != 0) return 0;
  size_t g = bytes / 16;
  if (g > 32 || (g & (g - 1)) != 0) return 0;
  return (int)g;
}

bool config_ok(const pilot_refine_config* c) {
  if (!c || c->n_levels < 1 || c->n_levels > PILOT_MAX_LEVELS) return false;
  if (c->feat_dtype != PILOT_F32 && c->feat_dtype != PILOT_BF16 && c->feat_dtype != PILOT_F16) return false;
  if (c->max_hypotheses < 1 || c->max_points < 1 || c->max_total_iters < 0) return false;
  for (int l = 0; l < c->n_levels; ++l)
    if (c->width[l] < 2 || c->height[l] < 2 || c->channels[l] < 1) return false;
  return true;
}

struct WsLayout { size_t state, counters, partials, total; int max_chunks; };

WsLayout ws_layout(const pilot_refine_config* c) {
  WsLayout w;
  w.max_chunks = (c->max_points + kMinChunk - 1) / kMinChunk;
  size_t o = 0;
  w.state = o;    o = align_up(o + sizeof(HypState) * (size_t)c->max_hypotheses, 256);
  w.counters = o; o = align_up(o + sizeof(unsigned) * (size_t)c->max_hypotheses, 256);
  w.partials = o; o = align_up(o + sizeof(float) * kNacc * (size_t)c->max_hypotheses * (size_t)w.max_chunks, 256);
  w.total = o;
  return w;
}

typedef void (*pass_fn)(const PassArgs);

template <class T, bool CEN>
pass_fn pick_g(int g) {
  switch (g) {
    case 1: return photo_pass_kernel<T, 1, CEN>;
    case 2: return photo_pass_kernel<T, 2, CEN>;
    case 4: return photo_pass_kernel<T, 4, CEN>;
    case 8: return photo_pass_kernel<T, 8, CEN>;
    case 16: return photo_pass_kernel<T, 16, CEN>;
    case 32: return photo_pass_kernel<T, 32, CEN>;
  }
  return nullptr;
}

template <bool CEN>
pass_fn pick_t(pilot_dtype d, int g) {
  switch (d) {
    case PILOT_F32: return pick_g<F32Tag, CEN>(g);
    case PILOT_BF16: return pick_g<BF16Tag, CEN>(g);
    case PILOT_F16: return pick_g<F16Tag, CEN>(g);
  }
  return nullptr;
}

pass_fn pick_kernel(pilot_dtype d, int g, int grad_mode) {
  return grad_mode == PILOT_GRAD_CENTRAL_SAMPLED ? pick_t<true>(d, g) : pick_t<false>(d, g);
}

int choose_chunk(const pilot_refine_handle* h, int n_hyp, int n_points) {
  if (h->chunk_override > 0) return h->chunk_override;
  // enough CTAs for ~4 waves at 2 CTAs/SM, chunks of 256..2048 anchors
  long want = 8L * h->sm_count;
  int chunk = 2048;
  while (chunk > kMinChunk && (long)n_hyp * ((n_points + chunk - 1) / chunk) < want) chunk >>= 1;
  return chunk;
}

}  // namespace

extern "C" {

size_t pilot_refine_workspace_bytes(const pilot_refine_config* cfg) {
  if (!config_ok(cfg)) return 0;
  return ws_layout(cfg).total;
}

int pilot_refine_create(const pilot_refine_config* cfg, pilot_refine_handle** out) {
  if (!out) return PILOT_ERR_ARG;
  *out = nullptr;
  if (!config_ok(cfg)) return PILOT_ERR_ARG;
  for (int l = 0; l < cfg->n_levels; ++l)
    if (lanes_per_unit(cfg->channels[l], cfg->feat_dtype) == 0) return PILOT_ERR_UNSUPPORTED;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) return PILOT_ERR_CUDA;
  int prev = 0;
  cudaGetDevice(&prev);
  if (cudaSetDevice(cfg->device) != cudaSuccess) return PILOT_ERR_CUDA;
  WsLayout w = ws_layout(cfg);
  pilot_refine_handle* h = new pilot_refine_handle();
  h->cfg = *cfg;
  h->max_chunks = w.max_chunks;
  h->chunk_override = 0;
  h->last_launches = 0;
  h->host_mode = false; h->stage = nullptr; h->stage_bytes = 0; h->max_dsm_w = h->max_dsm_h = 0;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess) { delete h; cudaSetDevice(prev); return PILOT_ERR_CUDA; }
  h->sm_count = prop.multiProcessorCount;
  if (cfg->workspace_dev) {
    if (cfg->workspace_bytes < w.total) { delete h; cudaSetDevice(prev); return PILOT_ERR_WORKSPACE; }
    h->ws = static_cast<char*>(cfg->workspace_dev);
    h->ws_bytes = cfg->workspace_bytes;
    h->owns_ws = false;
  } else {
    void* p = nullptr;
    if (cudaMalloc(&p, w.total) != cudaSuccess) { delete h; cudaSetDevice(prev); return PILOT_ERR_CUDA; }
    h->ws = static_cast<char*>(p);
    h->ws_bytes = w.total;
    h->owns_ws = true;
  }
  cudaSetDevice(prev);
  *out = h;
  return PILOT_OK;
}

int pilot_refine_destroy(pilot_refine_handle* h) {
  if (!h) return PILOT_OK;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(h->cfg.device);
  if (h->owns_ws && h->ws) cudaFree(h->ws);
  if (h->stage) cudaFree(h->stage);
  cudaSetDevice(prev);
  delete h;
  return PILOT_OK;
}

int pilot_refine_set_chunk(pilot_refine_handle* h, int chunk) {
  if (!h || chunk < 0 || (chunk % kMinChunk) != 0) return PILOT_ERR_ARG;
  h->chunk_override = chunk;
  return PILOT_OK;
}

int pilot_refine_last_launches(const pilot_refine_handle* h) { return h ? h->last_launches : 0; }

int pilot_refine_run(pilot_refine_handle* h, const pilot_refine_inputs* in, const pilot_refine_params* p,
                     const pilot_refine_outputs* out, void* cuda_stream) {
  if (!h) return PILOT_ERR_ARG;
  return pilot_refine_run_levels(h, in, p, out, 0, h->cfg.n_levels, cuda_stream);
}

int pilot_refine_run_levels(pilot_refine_handle* h, const pilot_refine_inputs* in, const pilot_refine_params* p,
                            const pilot_refine_outputs* out, int level_begin, int level_end, void* cuda_stream) {
  if (!h || !in || !p || !out) return PILOT_ERR_ARG;
  const pilot_refine_config& c = h->cfg;
  if (level_begin < 0 || level_begin >= level_end || level_end > c.n_levels) return PILOT_ERR_ARG;
  if (in->n_hypotheses < 0) return PILOT_ERR_ARG;
  if (in->n_hypotheses > c.max_hypotheses) return PILOT_ERR_UNSUPPORTED;
  int total_iters = 0;
  for (int l = 0; l < c.n_levels; ++l) {
    if (in->n_points[l] < 0 || p->iters[l] < 0) return PILOT_ERR_ARG;
    total_iters += p->iters[l];
    if (l < level_begin || l >= level_end) continue;       // pointers of levels outside the range are not read
    if (in->n_points[l] > c.max_points) return PILOT_ERR_UNSUPPORTED;
    if (!in->query_feat_dev[l]) return PILOT_ERR_ARG;
    if (in->n_points[l] > 0 && (!in->points_dev[l] || !in->ref_feat_dev[l])) return PILOT_ERR_ARG;
    if (((uintptr_t)in->query_feat_dev[l] | (uintptr_t)in->ref_feat_dev[l] | (uintptr_t)in->points_dev[l]) & 15) return PILOT_ERR_ARG;
  }
  if (total_iters > c.max_total_iters) return PILOT_ERR_UNSUPPORTED;
  if (p->grad_mode != PILOT_GRAD_BILINEAR_EXACT && p->grad_mode != PILOT_GRAD_CENTRAL_SAMPLED) return PILOT_ERR_ARG;
  if (p->loss < PILOT_LOSS_L2 || p->loss > PILOT_LOSS_CAUCHY) return PILOT_ERR_ARG;
  if (p->range_mode < PILOT_RANGE_OFF || p->range_mode > PILOT_RANGE_MARCH) return PILOT_ERR_ARG;
  if (p->range_mode == PILOT_RANGE_MARCH && (p->march_steps < 1 || p->bisect_steps < 0)) return PILOT_ERR_ARG;
  if (p->range_mode != PILOT_RANGE_OFF && p->w_range > 0.f && in->dsm_dev && (in->dsm_width < 2 || in->dsm_height < 2 || !(in->dsm_gsd > 0.f)))
    return PILOT_ERR_ARG;
  h->last_launches = 0;
  if (in->n_hypotheses == 0) return PILOT_OK;
  if (!in->init_poses_dev) return PILOT_ERR_ARG;

  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != c.device && cudaSetDevice(c.device) != cudaSuccess) return PILOT_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  WsLayout w = ws_layout(&c);
  PassArgs A;
  memset(&A, 0, sizeof A);
  A.prm = *p;
  for (int i = 0; i < 3; ++i) { A.gw[i] = in->gravity_world[i]; A.gi[i] = in->gravity_imu[i]; A.ray[i] = in->range_ray_cam[i]; }
  A.range_meas = in->range_meas;
  A.dsm = in->dsm_dev; A.dsm_w = in->dsm_width; A.dsm_h = in->dsm_height;
  A.dsm_ox = in->dsm_origin_x; A.dsm_oy = in->dsm_origin_y; A.dsm_gsd = in->dsm_gsd;
  A.n_hyp = in->n_hypotheses; A.level_end = level_end;
  A.state = reinterpret_cast<HypState*>(h->ws + w.state);
  A.counters = reinterpret_cast<unsigned*>(h->ws + w.counters);
  A.partials = reinterpret_cast<float*>(h->ws + w.partials);
  A.out = *out;

  int launches = 0;
  init_state_kernel<<<(A.n_hyp + 127) / 128, 128, 0, st>>>(A.state, A.counters, in->init_poses_dev, A.n_hyp, (double)p->lambda_init,
                                                                  level_begin);
  ++launches;
  int rec_base = 0;
  for (int l = 0; l < level_end; ++l) {
    if (l < level_begin) { rec_base += p->iters[l]; continue; }
    LevelArgs& L = A.lv;
    L.feat = in->query_feat_dev[l]; L.conf = in->query_conf_dev[l];
    L.points = reinterpret_cast<const float4*>(in->points_dev[l]); L.ref = in->ref_feat_dev[l];
    L.fx = in->intrinsics[l][0]; L.fy = in->intrinsics[l][1]; L.cx = in->intrinsics[l][2]; L.cy = in->intrinsics[l][3];
    L.W = c.width[l]; L.H = c.height[l]; L.C = c.channels[l]; L.N = in->n_points[l];
    A.level = l; A.iters = p->iters[l]; A.rec_base = rec_base;
    A.chunk = choose_chunk(h, A.n_hyp, L.N);
    A.n_chunks = L.N > 0 ? (L.N + A.chunk - 1) / A.chunk : 1;
    if (A.n_chunks > h->max_chunks) { A.chunk = kMinChunk; A.n_chunks = (L.N + kMinChunk - 1) / kMinChunk; }
    pass_fn fn = pick_kernel(c.feat_dtype, lanes_per_unit(L.C, c.feat_dtype), p->grad_mode);
    dim3 grid((unsigned)A.n_hyp, (unsigned)A.n_chunks);
    for (int pass = 0; pass <= p->iters[l]; ++pass) {
      A.pass = pass;
      fn<<<grid, kThreads, 0, st>>>(A);
      ++launches;
    }
    rec_base += p->iters[l];
  }
  h->last_launches = launches;
  cudaError_t e = cudaGetLastError();
  if (prev != c.device) cudaSetDevice(prev);
  return e == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

}  // extern "C"

// ====================================================================== host-buffer path (e2e)

namespace {

struct StageLayout {
  size_t feat[PILOT_MAX_LEVELS], conf[PILOT_MAX_LEVELS], pts[PILOT_MAX_LEVELS], ref[PILOT_MAX_LEVELS];
  size_t poses, dsm, o_poses, o_cost, o_nvalid, o_status, o_ih, o_ig, o_ic, o_il, total;
};

StageLayout stage_layout(const pilot_refine_config* c, int dsm_w, int dsm_h) {
  StageLayout s;
  size_t o = 0, es = elem_size(c->feat_dtype);
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
  for (int l = 0; l < PILOT_MAX_LEVELS; ++l) {
    bool on = l < c->n_levels;
    size_t px = on ? (size_t)c->width[l] * c->height[l] : 0;
    s.feat[l] = take(px * (on ? c->channels[l] : 0) * es);
    s.conf[l] = take(px * 4);
    s.pts[l] = take(on ? (size_t)c->max_points * 16 : 0);
    s.ref[l] = take(on ? (size_t)c->max_points * c->channels[l] * es : 0);
  }
  size_t H = (size_t)c->max_hypotheses, T = (size_t)c->max_total_iters;
  s.poses = take(H * 48);
  s.dsm = take((size_t)dsm_w * dsm_h * 4);
  s.o_poses = take(H * 48); s.o_cost = take(H * 4); s.o_nvalid = take(H * 4); s.o_status = take(H * 4);
  s.o_ih = take(T * H * 144); s.o_ig = take(T * H * 24); s.o_ic = take(T * H * 4); s.o_il = take(T * H * 4);
  s.total = o;
  return s;
}

}  // namespace

extern "C" {

int pilot_refine_create_host(const pilot_refine_config* cfg, int max_dsm_width, int max_dsm_height,
                             pilot_refine_handle** out) {
  if (!out) return PILOT_ERR_ARG;
  *out = nullptr;
  if (!cfg || cfg->workspace_dev || max_dsm_width < 0 || max_dsm_height < 0) return PILOT_ERR_ARG;
  int rc = pilot_refine_create(cfg, out);
  if (rc != PILOT_OK) return rc;
  pilot_refine_handle* h = *out;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(cfg->device);
  StageLayout s = stage_layout(cfg, max_dsm_width, max_dsm_height);
  void* p = nullptr;
  cudaError_t e = cudaMalloc(&p, s.total);
  cudaSetDevice(prev);
  if (e != cudaSuccess) { pilot_refine_destroy(h); *out = nullptr; return PILOT_ERR_CUDA; }
  h->stage = static_cast<char*>(p);
  h->stage_bytes = s.total;
  h->host_mode = true;
  h->max_dsm_w = max_dsm_width; h->max_dsm_h = max_dsm_height;
  return PILOT_OK;
}

int pilot_refine_run_host(pilot_refine_handle* h, const pilot_refine_inputs* in, const pilot_refine_params* p,
                          const pilot_refine_outputs* out, void* cuda_stream) {
  if (!h || !in || !p || !out || !h->host_mode) return PILOT_ERR_ARG;
  const pilot_refine_config& c = h->cfg;
  if (in->n_hypotheses < 0 || in->n_hypotheses > c.max_hypotheses) return in->n_hypotheses < 0 ? PILOT_ERR_ARG : PILOT_ERR_UNSUPPORTED;
  int T = 0;
  for (int l = 0; l < c.n_levels; ++l) {
    if (in->n_points[l] < 0 || p->iters[l] < 0) return PILOT_ERR_ARG;
    if (in->n_points[l] > c.max_points) return PILOT_ERR_UNSUPPORTED;
    T += p->iters[l];
  }
  if (T > c.max_total_iters) return PILOT_ERR_UNSUPPORTED;
  if (in->dsm_dev && ((size_t)in->dsm_width * in->dsm_height > (size_t)h->max_dsm_w * h->max_dsm_h)) return PILOT_ERR_UNSUPPORTED;
  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != c.device && cudaSetDevice(c.device) != cudaSuccess) return PILOT_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  StageLayout s = stage_layout(&c, h->max_dsm_w, h->max_dsm_h);
  size_t es = elem_size(c.feat_dtype), H = (size_t)in->n_hypotheses;
  pilot_refine_inputs din = *in;
  bool ok = true;
  auto up = [&](size_t at, const void* src, size_t bytes) -> void* {
    if (!src || bytes == 0) return nullptr;
    ok = ok && cudaMemcpyAsync(h->stage + at, src, bytes, cudaMemcpyHostToDevice, st) == cudaSuccess;
    return h->stage + at;
  };
  for (int l = 0; l < c.n_levels; ++l) {
    size_t px = (size_t)c.width[l] * c.height[l], N = (size_t)in->n_points[l];
    din.query_feat_dev[l] = up(s.feat[l], in->query_feat_dev[l], px * c.channels[l] * es);
    din.query_conf_dev[l] = static_cast<const float*>(up(s.conf[l], in->query_conf_dev[l], px * 4));
    din.points_dev[l] = static_cast<const float*>(up(s.pts[l], in->points_dev[l], N * 16));
    din.ref_feat_dev[l] = up(s.ref[l], in->ref_feat_dev[l], N * c.channels[l] * es);
  }
  din.init_poses_dev = static_cast<const float*>(up(s.poses, in->init_poses_dev, H * 48));
  din.dsm_dev = static_cast<const float*>(up(s.dsm, in->dsm_dev, (size_t)in->dsm_width * in->dsm_height * 4));
  pilot_refine_outputs dout;
  dout.poses_dev = out->poses_dev ? reinterpret_cast<float*>(h->stage + s.o_poses) : nullptr;
  dout.cost_dev = out->cost_dev ? reinterpret_cast<float*>(h->stage + s.o_cost) : nullptr;
  dout.n_valid_dev = out->n_valid_dev ? reinterpret_cast<int*>(h->stage + s.o_nvalid) : nullptr;
  dout.status_dev = out->status_dev ? reinterpret_cast<unsigned*>(h->stage + s.o_status) : nullptr;
  dout.iter_hessian_dev = out->iter_hessian_dev ? reinterpret_cast<float*>(h->stage + s.o_ih) : nullptr;
  dout.iter_gradient_dev = out->iter_gradient_dev ? reinterpret_cast<float*>(h->stage + s.o_ig) : nullptr;
  dout.iter_cost_dev = out->iter_cost_dev ? reinterpret_cast<float*>(h->stage + s.o_ic) : nullptr;
  dout.iter_lambda_dev = out->iter_lambda_dev ? reinterpret_cast<float*>(h->stage + s.o_il) : nullptr;
  int rc = ok ? pilot_refine_run(h, &din, p, &dout, cuda_stream) : PILOT_ERR_CUDA;
  if (rc == PILOT_OK) {
    auto down = [&](void* dst, const void* src, size_t bytes) {
      if (dst && bytes) ok = ok && cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st) == cudaSuccess;
    };
    down(out->poses_dev, dout.poses_dev, H * 48);
    down(out->cost_dev, dout.cost_dev, H * 4);
    down(out->n_valid_dev, dout.n_valid_dev, H * 4);
    down(out->status_dev, dout.status_dev, H * 4);
    down(out->iter_hessian_dev, dout.iter_hessian_dev, (size_t)T * H * 144);
    down(out->iter_gradient_dev, dout.iter_gradient_dev, (size_t)T * H * 24);
    down(out->iter_cost_dev, dout.iter_cost_dev, (size_t)T * H * 4);
    down(out->iter_lambda_dev, dout.iter_lambda_dev, (size_t)T * H * 4);
    ok = ok && cudaStreamSynchronize(st) == cudaSuccess;
    if (!ok) rc = PILOT_ERR_CUDA;
  }
  if (prev != c.device) cudaSetDevice(prev);
  return rc;
}

}  // extern "C"
