/*
 * pilot_oracle.c — double-precision CPU oracle (TEST INFRASTRUCTURE; see pilot_oracle.h).
 * Scalar loops, no blocking, no fusion: each function is the paper's definition written out.
 * Build: gcc -O2 -std=c11 -fPIC -shared [-fopenmp] -o libpilot_oracle.so pilot_oracle.c -lm
 */
#include "pilot_oracle.h"

#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ element decoding */

static double decode_bf16(uint16_t h) {
  uint32_t u = ((uint32_t)h) << 16; /* bf16 = top half of an IEEE fp32 */
  float f;
  memcpy(&f, &u, 4);
  return (double)f;
}

static double decode_f16(uint16_t h) {
  int sign = (h >> 15) & 1, e = (h >> 10) & 31, m = h & 1023;
  double v;
  if (e == 0) v = ldexp((double)m, -24);                 /* subnormal */
  else if (e == 31) v = m ? NAN : INFINITY;
  else v = ldexp((double)(m + 1024), e - 25);
  return sign ? -v : v;
}

static double feat_at(const void* base, pilot_dtype dt, size_t idx) {
  switch (dt) {
    case PILOT_F32:  return (double)((const float*)base)[idx];
    case PILOT_BF16: return decode_bf16(((const uint16_t*)base)[idx]);
    case PILOT_F16:  return decode_f16(((const uint16_t*)base)[idx]);
  }
  return NAN;
}

/* ------------------------------------------------------------------ robust losses (Eq.2, Eq.7) */

void pilot_oracle_loss(int loss, double x, double scale, double* rho, double* drho) {
  double r = x, d = 1.0;
  if (scale > 0.0) {
    double s2 = scale * scale;
    if (loss == PILOT_LOSS_HUBER) {          /* Huber on sqrt(x): quadratic inside delta, linear outside */
      if (x > s2) { double sq = sqrt(x); r = 2.0 * scale * sq - s2; d = scale / sq; }
    } else if (loss == PILOT_LOSS_CAUCHY) {
      r = s2 * log1p(x / s2);
      d = 1.0 / (1.0 + x / s2);
    }
  }
  if (rho) *rho = r;
  if (drho) *drho = d;
}

/* ------------------------------------------------------------------ small 3x3 helpers */

static void mat3_mul(const double A[9], const double B[9], double C[9]) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      double s = 0.0;
      for (int k = 0; k < 3; ++k) s += A[3 * i + k] * B[3 * k + j];
      C[3 * i + j] = s;
    }
}
static void mat3_vec(const double A[9], const double x[3], double y[3]) {
  for (int i = 0; i < 3; ++i) y[i] = A[3 * i] * x[0] + A[3 * i + 1] * x[1] + A[3 * i + 2] * x[2];
}
static void mat3T_vec(const double A[9], const double x[3], double y[3]) {
  for (int i = 0; i < 3; ++i) y[i] = A[i] * x[0] + A[3 + i] * x[1] + A[6 + i] * x[2];
}
static void skew(const double a[3], double S[9]) {
  S[0] = 0;     S[1] = -a[2]; S[2] = a[1];
  S[3] = a[2];  S[4] = 0;     S[5] = -a[0];
  S[6] = -a[1]; S[7] = a[0];  S[8] = 0;
}

/* ------------------------------------------------------------------ SE(3) exp (Eq.9) */

void pilot_oracle_se3_exp(const double xi[6], double E[9], double V[9]) {
  const double* phi = xi + 3;
  double th2 = phi[0] * phi[0] + phi[1] * phi[1] + phi[2] * phi[2];
  double th = sqrt(th2);
  double A, B, Cc; /* sin(th)/th, (1-cos th)/th^2, (th - sin th)/th^3 */
  if (th < 1e-4) {
    A = 1.0 - th2 / 6.0 + th2 * th2 / 120.0;
    B = 0.5 - th2 / 24.0 + th2 * th2 / 720.0;
    Cc = 1.0 / 6.0 - th2 / 120.0 + th2 * th2 / 5040.0;
  } else {
    A = sin(th) / th;
    B = (1.0 - cos(th)) / th2;
    Cc = (th - sin(th)) / (th2 * th);
  }
  double K[9], K2[9];
  skew(phi, K);
  mat3_mul(K, K, K2);
  for (int i = 0; i < 9; ++i) {
    double I = (i % 4 == 0) ? 1.0 : 0.0;
    E[i] = I + A * K[i] + B * K2[i];   /* Rodrigues */
    V[i] = I + B * K[i] + Cc * K2[i];
  }
}

void pilot_oracle_retract(const double R_cw[9], const double C[3], const double xi[6],
                          double R_out[9], double C_out[3]) {
  /* T_cw <- exp(xi) T_cw with T_cw = [R_cw | t], t = -R_cw C:
   *   R' = E R_cw ; t' = E t + V rho ; C' = -R'^T t' = C - R_cw^T E^T V rho.            */
  double E[9], V[9], Vr[3], EtVr[3], d[3], Rn[9];
  pilot_oracle_se3_exp(xi, E, V);
  mat3_vec(V, xi, Vr);
  mat3T_vec(E, Vr, EtVr);
  mat3T_vec(R_cw, EtVr, d);
  mat3_mul(E, R_cw, Rn);
  for (int i = 0; i < 9; ++i) R_out[i] = Rn[i];
  for (int i = 0; i < 3; ++i) C_out[i] = C[i] - d[i];
}

/* ------------------------------------------------------------------ 6x6 Cholesky (Eq.8) */

int pilot_oracle_chol_solve6(const double A[36], const double b[6], double x[6]) {
  double L[36];
  memset(L, 0, sizeof L);
  for (int i = 0; i < 6; ++i) {
    for (int j = 0; j <= i; ++j) {
      double s = A[6 * i + j];
      for (int k = 0; k < j; ++k) s -= L[6 * i + k] * L[6 * j + k];
      if (i == j) {
        if (!(s > 0.0) || !isfinite(s)) return 0;
        L[6 * i + i] = sqrt(s);
      } else {
        L[6 * i + j] = s / L[6 * j + j];
      }
    }
  }
  double y[6];
  for (int i = 0; i < 6; ++i) {
    double s = b[i];
    for (int k = 0; k < i; ++k) s -= L[6 * i + k] * y[k];
    y[i] = s / L[6 * i + i];
  }
  for (int i = 5; i >= 0; --i) {
    double s = y[i];
    for (int k = i + 1; k < 6; ++k) s -= L[6 * k + i] * x[k];
    x[i] = s / L[6 * i + i];
  }
  for (int i = 0; i < 6; ++i)
    if (!isfinite(x[i])) return 0;
  return 1;
}

/* ------------------------------------------------------------------ DSM sample (Eq.6) */

int pilot_oracle_dsm_sample(const pilot_refine_inputs* in, double x, double y,
                            double* z, double* dzdx, double* dzdy) {
  double gsd = (double)in->dsm_gsd;
  double gx = (x - (double)in->dsm_origin_x) / gsd;
  double gy = (y - (double)in->dsm_origin_y) / gsd;
  if (!isfinite(gx) || !isfinite(gy)) return 0;
  double fx0 = floor(gx), fy0 = floor(gy);
  if (fx0 < 0.0 || fy0 < 0.0 || fx0 > (double)(in->dsm_width - 2) || fy0 > (double)(in->dsm_height - 2))
    return 0;
  int ix = (int)fx0, iy = (int)fy0;
  double a = gx - fx0, b = gy - fy0;
  const float* D = in->dsm_dev;
  size_t W = (size_t)in->dsm_width;
  double d00 = D[(size_t)iy * W + ix], d10 = D[(size_t)iy * W + ix + 1];
  double d01 = D[(size_t)(iy + 1) * W + ix], d11 = D[(size_t)(iy + 1) * W + ix + 1];
  if (z) *z = (1 - b) * ((1 - a) * d00 + a * d10) + b * ((1 - a) * d01 + a * d11);
  if (dzdx) *dzdx = ((1 - b) * (d10 - d00) + b * (d11 - d01)) / gsd;
  if (dzdy) *dzdy = ((1 - a) * (d01 - d00) + a * (d11 - d10)) / gsd;
  return 1;
}

/* ------------------------------------------------------------------ photo term, one point (Eq.1) */

static void tap(const pilot_refine_config* cfg, const pilot_refine_inputs* in, int level,
                int x, int y, int c, double* out) {
  size_t W = (size_t)cfg->width[level], C = (size_t)cfg->channels[level];
  *out = feat_at(in->query_feat_dev[level], cfg->feat_dtype, ((size_t)y * W + (size_t)x) * C + (size_t)c);
}

static int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* central-difference gradient maps Dx, Dy at integer pixel (x,y), replicate border (reading A7) */
static void central_diff(const pilot_refine_config* cfg, const pilot_refine_inputs* in, int level,
                         int x, int y, int c, double* dx, double* dy) {
  int W = cfg->width[level], H = cfg->height[level];
  double xp, xm, yp, ym;
  tap(cfg, in, level, clampi(x + 1, 0, W - 1), y, c, &xp);
  tap(cfg, in, level, clampi(x - 1, 0, W - 1), y, c, &xm);
  tap(cfg, in, level, x, clampi(y + 1, 0, H - 1), c, &yp);
  tap(cfg, in, level, x, clampi(y - 1, 0, H - 1), c, &ym);
  *dx = 0.5 * (xp - xm);
  *dy = 0.5 * (yp - ym);
}

int pilot_oracle_photo_point(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                             const pilot_refine_params* p, int level,
                             const double R_cw[9], const double C[3], int j,
                             double uv[2], double* f, double* gx, double* gy, double* r,
                             double Juv[12], double* w) {
  const float* P = in->points_dev[level] + 4 * (size_t)j;
  double d[3] = {(double)P[0] - C[0], (double)P[1] - C[1], (double)P[2] - C[2]};
  double pc[3];
  mat3_vec(R_cw, d, pc);                               /* p = R_cw (P_j - C) = T~^-1 P_j */
  double X = pc[0], Y = pc[1], Z = pc[2];
  if (!(Z > (double)p->z_near)) return 0;
  double fx = in->intrinsics[level][0], fy = in->intrinsics[level][1];
  double cx = in->intrinsics[level][2], cy = in->intrinsics[level][3];
  double u = fx * X / Z + cx, v = fy * Y / Z + cy;     /* pinhole pi(K_l, ., .) */
  if (!isfinite(u) || !isfinite(v)) return 0;
  int W = cfg->width[level], H = cfg->height[level], Cn = cfg->channels[level];
  double fx0 = floor(u), fy0 = floor(v);
  if (fx0 < 0.0 || fy0 < 0.0 || fx0 + 1.0 > (double)(W - 1) || fy0 + 1.0 > (double)(H - 1)) return 0;
  int x0 = (int)fx0, y0 = (int)fy0;
  double a = u - fx0, b = v - fy0;
  if (uv) { uv[0] = u; uv[1] = v; }
  for (int c = 0; c < Cn; ++c) {
    double f00, f10, f01, f11;
    tap(cfg, in, level, x0, y0, c, &f00);
    tap(cfg, in, level, x0 + 1, y0, c, &f10);
    tap(cfg, in, level, x0, y0 + 1, c, &f01);
    tap(cfg, in, level, x0 + 1, y0 + 1, c, &f11);
    double fv = (1 - b) * ((1 - a) * f00 + a * f10) + b * ((1 - a) * f01 + a * f11);
    double gxv, gyv;
    if (p->grad_mode == PILOT_GRAD_BILINEAR_EXACT) {
      gxv = (1 - b) * (f10 - f00) + b * (f11 - f01);
      gyv = (1 - a) * (f01 - f00) + a * (f11 - f10);
    } else {
      double dx00, dy00, dx10, dy10, dx01, dy01, dx11, dy11;
      central_diff(cfg, in, level, x0, y0, c, &dx00, &dy00);
      central_diff(cfg, in, level, x0 + 1, y0, c, &dx10, &dy10);
      central_diff(cfg, in, level, x0, y0 + 1, c, &dx01, &dy01);
      central_diff(cfg, in, level, x0 + 1, y0 + 1, c, &dx11, &dy11);
      gxv = (1 - b) * ((1 - a) * dx00 + a * dx10) + b * ((1 - a) * dx01 + a * dx11);
      gyv = (1 - b) * ((1 - a) * dy00 + a * dy10) + b * ((1 - a) * dy01 + a * dy11);
    }
    if (f) f[c] = fv;
    if (gx) gx[c] = gxv;
    if (gy) gy[c] = gyv;
    if (r) r[c] = fv - feat_at(in->ref_feat_dev[level], cfg->feat_dtype, (size_t)j * (size_t)Cn + (size_t)c);
  }
  if (Juv) {
    double iz = 1.0 / Z, iz2 = iz * iz;
    Juv[0] = fx * iz; Juv[1] = 0.0;     Juv[2] = -fx * X * iz2;
    Juv[3] = -fx * X * Y * iz2; Juv[4] = fx * (1.0 + X * X * iz2); Juv[5] = -fx * Y * iz;
    Juv[6] = 0.0;     Juv[7] = fy * iz; Juv[8] = -fy * Y * iz2;
    Juv[9] = -fy * (1.0 + Y * Y * iz2); Juv[10] = fy * X * Y * iz2; Juv[11] = fy * X * iz;
  }
  if (w) {
    double wq = 1.0;
    const float* Q = in->query_conf_dev[level];
    if (Q) {
      size_t Ws = (size_t)W;
      double q00 = Q[(size_t)y0 * Ws + x0], q10 = Q[(size_t)y0 * Ws + x0 + 1];
      double q01 = Q[(size_t)(y0 + 1) * Ws + x0], q11 = Q[(size_t)(y0 + 1) * Ws + x0 + 1];
      wq = (1 - b) * ((1 - a) * q00 + a * q10) + b * ((1 - a) * q01 + a * q11);
    }
    *w = (double)P[3] * wq;
  }
  return 1;
}

/* ------------------------------------------------------------------ gravity prior (Eq.3) */

void pilot_oracle_gravity(const pilot_refine_inputs* in, const double R_cw[9],
                          double r[3], double J[18]) {
  double gw[3] = {in->gravity_world[0], in->gravity_world[1], in->gravity_world[2]};
  double e[3], S[9];
  mat3_vec(R_cw, gw, e);                               /* R(T~)^T gamma^W, R(T~) = R_wc = R_cw^T */
  for (int i = 0; i < 3; ++i) r[i] = e[i] - (double)in->gravity_imu[i];
  if (J) {
    skew(e, S);                                        /* d(E e)/dphi = -[e]x ; translation does nothing */
    for (int i = 0; i < 3; ++i)
      for (int k = 0; k < 3; ++k) { J[6 * i + k] = 0.0; J[6 * i + 3 + k] = -S[3 * i + k]; }
  }
}

/* ------------------------------------------------------------------ range prior (Eq.4-6; ray-march) */

static double height_above(const pilot_refine_inputs* in, const double C[3], const double wr[3], double t) {
  double z;
  double x = C[0] + t * wr[0], y = C[1] + t * wr[1];
  if (!pilot_oracle_dsm_sample(in, x, y, &z, NULL, NULL)) return INFINITY; /* off the map counts as above */
  return C[2] + t * wr[2] - z;
}

int pilot_oracle_range(const pilot_refine_inputs* in, const pilot_refine_params* p,
                       const double R_cw[9], const double C[3],
                       double* r, double J[6], double* d_hit) {
  if (p->range_mode == PILOT_RANGE_OFF || !in->dsm_dev) return 0;
  double v[3] = {in->range_ray_cam[0], in->range_ray_cam[1], in->range_ray_cam[2]};
  double wr[3];
  mat3T_vec(R_cw, v, wr);                              /* world ray R(T~) v */
  double dist, res, ndotw = 1.0;
  double dm = (double)in->range_meas;
  if (p->range_mode == PILOT_RANGE_HEIGHT) {
    dist = dm;
  } else {
    int steps = p->march_steps;
    double tfar = (double)p->march_tfar_scale * dm, dt = tfar / (double)steps;
    int found = -1;
    double fprev = height_above(in, C, wr, 0.0);
    for (int i = 0; i < steps; ++i) {
      double fnext = height_above(in, C, wr, (double)(i + 1) * dt);
      if (fprev > 0.0 && fnext <= 0.0) { found = i; break; }
      fprev = fnext;
    }
    if (found < 0) return 0;
    double lo = (double)found * dt, hi = (double)(found + 1) * dt;
    for (int k = 0; k < p->bisect_steps; ++k) {
      double mid = 0.5 * (lo + hi);
      if (height_above(in, C, wr, mid) > 0.0) lo = mid; else hi = mid;
    }
    double flo = height_above(in, C, wr, lo), fhi = height_above(in, C, wr, hi);
    if (isfinite(flo) && isfinite(fhi) && flo - fhi > 0.0) dist = lo + (hi - lo) * flo / (flo - fhi);
    else dist = hi;
  }
  double q[3] = {dist * v[0], dist * v[1], dist * v[2]};
  double Pw[3] = {C[0] + dist * wr[0], C[1] + dist * wr[1], C[2] + dist * wr[2]};   /* Eq.(5) */
  double z, dzdx, dzdy;
  if (!pilot_oracle_dsm_sample(in, Pw[0], Pw[1], &z, &dzdx, &dzdy)) return 0;
  double n[3] = {-dzdx, -dzdy, 1.0};
  if (p->range_mode == PILOT_RANGE_HEIGHT) {
    res = Pw[2] - z;                                   /* Eq.(6) */
  } else {
    res = dist - dm;
    ndotw = n[0] * wr[0] + n[1] * wr[1] + n[2] * wr[2];
    if (!(fabs(ndotw) > 1e-12)) return 0;
  }
  if (r) *r = res;
  if (d_hit) *d_hit = dist;
  if (J) {
    /* dP/dxi = R_cw^T [ -I | [q]x ]  =>  row = n^T R_cw^T [ -I | [q]x ] */
    double m[3], Sq[9];
    mat3_vec(R_cw, n, m);                              /* m = R_cw n  (m^T = n^T R_cw^T) */
    skew(q, Sq);
    for (int k = 0; k < 3; ++k) {
      J[k] = -m[k];
      J[3 + k] = m[0] * Sq[k] + m[1] * Sq[3 + k] + m[2] * Sq[6 + k];
    }
    if (p->range_mode == PILOT_RANGE_MARCH)
      for (int k = 0; k < 6; ++k) J[k] = -J[k] / ndotw;
  }
  return 1;
}

/* ------------------------------------------------------------------ EVAL: total system (Eq.7, supp Eq.5-6) */

static void add_outer(double H[36], double g[6], const double J[6], double r, double wgt) {
  for (int a = 0; a < 6; ++a) {
    g[a] += wgt * J[a] * r;
    for (int b = a; b < 6; ++b) {                    /* upper triangle, mirrored: H = H^T exactly */
      double h = wgt * J[a] * J[b];
      H[6 * a + b] += h;
      if (b != a) H[6 * b + a] += h;
    }
  }
}

void pilot_oracle_eval(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                       const pilot_refine_params* p, int level, int which,
                       const double R_cw[9], const double C[3],
                       double H_out[36], double g_out[6], double* cost_out, int* n_valid_out,
                       double* g_abs_out, unsigned* flags_out) {
  double H[36], g[6], cost = 0.0, gabs = 0.0;
  unsigned flags = 0;
  int nvalid = 0;
  memset(H, 0, sizeof H);
  memset(g, 0, sizeof g);
  int Cn = cfg->channels[level];
  double* buf = (double*)malloc(sizeof(double) * 3 * (size_t)Cn);
  double *gx = buf, *gy = buf + Cn, *r = buf + 2 * Cn;

  if (which & 1) {
    for (int j = 0; j < in->n_points[level]; ++j) {
      double Juv[12], w;
      if (!pilot_oracle_photo_point(cfg, in, p, level, R_cw, C, j, NULL, NULL, gx, gy, r, Juv, &w)) continue;
      double s = 0.0, A11 = 0.0, A12 = 0.0, A22 = 0.0, b1 = 0.0, b2 = 0.0;
      for (int c = 0; c < Cn; ++c) {
        s += r[c] * r[c];
        A11 += gx[c] * gx[c]; A12 += gx[c] * gy[c]; A22 += gy[c] * gy[c];
        b1 += gx[c] * r[c];   b2 += gy[c] * r[c];
      }
      double rho, drho;
      pilot_oracle_loss(p->loss, w * s, (double)p->loss_scale, &rho, &drho);  /* rho(w ||r||^2), Eq.(2) */
      double omega = w * drho;
      const double* Ju = Juv;
      const double* Jv = Juv + 6;
      double gj[6], n2 = 0.0;
      for (int a = 0; a < 6; ++a) {
        gj[a] = omega * (Ju[a] * b1 + Jv[a] * b2);
        g[a] += gj[a];
        n2 += gj[a] * gj[a];
        for (int b = a; b < 6; ++b) {                /* upper triangle, mirrored: H = H^T exactly */
          double h = omega * (A11 * Ju[a] * Ju[b] + A12 * (Ju[a] * Jv[b] + Jv[a] * Ju[b]) + A22 * Jv[a] * Jv[b]);
          H[6 * a + b] += h;
          if (b != a) H[6 * b + a] += h;
        }
      }
      gabs += sqrt(n2);
      cost += rho;
      nvalid += 1;
    }
    if (nvalid < p->min_valid) { cost = INFINITY; flags |= PILOT_ORACLE_FEW_VALID; }
  }

  if ((which & 2) && p->w_gravity > 0.0f) {
    double rg[3], Jg[18], rho, drho;
    pilot_oracle_gravity(in, R_cw, rg, Jg);
    double x = rg[0] * rg[0] + rg[1] * rg[1] + rg[2] * rg[2];
    pilot_oracle_loss(p->loss, x, (double)p->gravity_scale, &rho, &drho);
    double wgt = (double)p->w_gravity * drho, gj[6] = {0, 0, 0, 0, 0, 0}, n2 = 0.0;
    for (int i = 0; i < 3; ++i) {
      add_outer(H, g, Jg + 6 * i, rg[i], wgt);
      for (int a = 0; a < 6; ++a) gj[a] += wgt * Jg[6 * i + a] * rg[i];
    }
    for (int a = 0; a < 6; ++a) n2 += gj[a] * gj[a];
    gabs += sqrt(n2);
    cost += (double)p->w_gravity * rho;
  }

  if ((which & 4) && p->range_mode != PILOT_RANGE_OFF && p->w_range > 0.0f) {
    double rr, Jr[6], rho, drho;
    if (pilot_oracle_range(in, p, R_cw, C, &rr, Jr, NULL)) {
      pilot_oracle_loss(p->loss, rr * rr, (double)p->range_scale, &rho, &drho);
      double wgt = (double)p->w_range * drho, n2 = 0.0;
      add_outer(H, g, Jr, rr, wgt);
      for (int a = 0; a < 6; ++a) n2 += (wgt * Jr[a] * rr) * (wgt * Jr[a] * rr);
      gabs += sqrt(n2);
      cost += (double)p->w_range * rho;
    } else {
      flags |= PILOT_ORACLE_RANGE_SKIP;
    }
  }
  free(buf);
  if (H_out) memcpy(H_out, H, sizeof H);
  if (g_out) memcpy(g_out, g, sizeof g);
  if (cost_out) *cost_out = cost;
  if (n_valid_out) *n_valid_out = nvalid;
  if (g_abs_out) *g_abs_out = gabs;
  if (flags_out) *flags_out = flags;
}

/* ------------------------------------------------------------------ the LM loop (Eq.8-9) */

typedef struct { double H[36], g[6], cost, gabs; int nvalid; unsigned flags; } sys_t;

static void eval_sys(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                     const pilot_refine_params* p, int level, const double R[9], const double C[3], sys_t* S) {
  pilot_oracle_eval(cfg, in, p, level, 7, R, C, S->H, S->g, &S->cost, &S->nvalid, &S->gabs, &S->flags);
}

static void pose_out(const double R_cw[9], const double C[3], double T[12]) {
  for (int i = 0; i < 3; ++i) {
    for (int k = 0; k < 3; ++k) T[4 * i + k] = R_cw[3 * k + i];  /* R_wc = R_cw^T */
    T[4 * i + 3] = C[i];
  }
}

static void run_one(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                    const pilot_refine_params* p, const pilot_refine_outputs* out,
                    const pilot_oracle_extra* ex, int m) {
  int Hn = in->n_hypotheses;
  const float* T0 = in->init_poses_dev + 12 * (size_t)m;
  double R[9], C[3];
  for (int i = 0; i < 3; ++i) {
    for (int k = 0; k < 3; ++k) R[3 * k + i] = (double)T0[4 * i + k];
    C[i] = (double)T0[4 * i + 3];
  }
  unsigned status = 0;
  double last_step = INFINITY;
  sys_t S;
  memset(&S, 0, sizeof S);
  int rec = 0;
  for (int l = 0; l < cfg->n_levels; ++l) {
    double lam = (double)p->lambda_init;
    last_step = INFINITY;
    eval_sys(cfg, in, p, l, R, C, &S);
    if (isnan(S.cost)) status |= PILOT_STATUS_NONFINITE;
    for (int k = 0; k < p->iters[l]; ++k, ++rec) {
      size_t ri = (size_t)rec * (size_t)Hn + (size_t)m;
      if (out->iter_hessian_dev) for (int i = 0; i < 36; ++i) out->iter_hessian_dev[36 * ri + i] = (float)S.H[i];
      if (out->iter_gradient_dev) for (int i = 0; i < 6; ++i) out->iter_gradient_dev[6 * ri + i] = (float)S.g[i];
      if (out->iter_cost_dev) out->iter_cost_dev[ri] = (float)S.cost;
      if (out->iter_lambda_dev) out->iter_lambda_dev[ri] = (float)lam;
      if (ex && ex->iter_gabs) ex->iter_gabs[ri] = S.gabs;
      if (ex && ex->iter_poses) pose_out(R, C, ex->iter_poses + 12 * ri);

      double A[36], dxi[6];
      memcpy(A, S.H, sizeof A);
      for (int i = 0; i < 6; ++i) {
        if (p->damp_mode == PILOT_DAMP_IDENTITY) A[7 * i] += lam;                       /* Eq.(8): lambda I */
        else A[7 * i] += lam * (S.H[7 * i] > 1e-12 ? S.H[7 * i] : 1e-12);
      }
      int ok = pilot_oracle_chol_solve6(A, S.g, dxi);
      if (!ok) {
        if (lam >= (double)p->lambda_max) status |= PILOT_STATUS_CHOL_FAIL;
        lam = fmin(lam * (double)p->lambda_up, (double)p->lambda_max);
        continue;
      }
      double n2 = 0.0;
      for (int i = 0; i < 6; ++i) { dxi[i] = -dxi[i]; n2 += dxi[i] * dxi[i]; }
      double Rn[9], Cn[3];
      pilot_oracle_retract(R, C, dxi, Rn, Cn);                                          /* Eq.(9) */
      sys_t Sn;
      eval_sys(cfg, in, p, l, Rn, Cn, &Sn);
      if (isnan(Sn.cost)) status |= PILOT_STATUS_NONFINITE;
      if (p->lm_mode == PILOT_LM_FIXED || Sn.cost < S.cost) {
        memcpy(R, Rn, sizeof R); memcpy(C, Cn, sizeof C);
        S = Sn;
        last_step = sqrt(n2);
        if (p->lm_mode == PILOT_LM_ADAPTIVE) lam = fmax(lam * (double)p->lambda_down, (double)p->lambda_min);
      } else {
        lam = fmin(lam * (double)p->lambda_up, (double)p->lambda_max);
      }
    }
  }
  if (S.flags & PILOT_ORACLE_FEW_VALID) status |= PILOT_STATUS_FEW_VALID;
  if (S.flags & PILOT_ORACLE_RANGE_SKIP) status |= PILOT_STATUS_RANGE_SKIP;
  double T[12];
  pose_out(R, C, T);
  if (out->poses_dev) for (int i = 0; i < 12; ++i) out->poses_dev[12 * (size_t)m + i] = (float)T[i];
  if (out->cost_dev) out->cost_dev[m] = (float)S.cost;
  if (out->n_valid_dev) out->n_valid_dev[m] = S.nvalid;
  if (out->status_dev) out->status_dev[m] = status;
  if (ex && ex->poses) memcpy(ex->poses + 12 * (size_t)m, T, sizeof T);
  if (ex && ex->cost) ex->cost[m] = S.cost;
  if (ex && ex->last_step) ex->last_step[m] = last_step;
}

int pilot_oracle_threads(int n_threads) {
#ifdef _OPENMP
  if (n_threads < 1) n_threads = 1;
  int mx = omp_get_num_procs();
  return n_threads > mx ? mx : n_threads;
#else
  (void)n_threads;
  return 1;
#endif
}

int pilot_oracle_run(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                     const pilot_refine_params* p, const pilot_refine_outputs* out,
                     const pilot_oracle_extra* extra,
                     int hyp_begin, int hyp_step, int n_threads) {
  if (!cfg || !in || !p || !out) return PILOT_ERR_ARG;
  if (cfg->n_levels < 1 || cfg->n_levels > PILOT_MAX_LEVELS) return PILOT_ERR_ARG;
  if (in->n_hypotheses < 0 || !in->init_poses_dev) return PILOT_ERR_ARG;
  if (hyp_step < 1 || hyp_begin < 0) return PILOT_ERR_ARG;
  for (int l = 0; l < cfg->n_levels; ++l) {
    if (!in->query_feat_dev[l] || (in->n_points[l] > 0 && (!in->points_dev[l] || !in->ref_feat_dev[l]))) return PILOT_ERR_ARG;
    if (p->iters[l] < 0) return PILOT_ERR_ARG;
  }
  int nt = pilot_oracle_threads(n_threads);
  (void)nt;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt)
#endif
  for (int m = hyp_begin; m < in->n_hypotheses; m += hyp_step) run_one(cfg, in, p, out, extra, m);
  return PILOT_OK;
}
