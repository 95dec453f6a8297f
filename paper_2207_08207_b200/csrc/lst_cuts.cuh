// lst_cuts.cuh -- the four selections of DESIGN.md section 1 ("SPEC"), device side.
//
// Typed from the SPEC, not from the oracle.  This translation unit is compiled with
// --fmad=false (no FMA contraction), default -prec-div / -prec-sqrt (IEEE), no -ftz, so every
// expression below is evaluated in binary32 round-to-nearest in the parenthesisation written.
// Comparisons are `!(value <= threshold)` -> reject, so a NaN rejects (reading 14).
#pragma once
#include <cuda_runtime.h>

namespace lst {

// Cut constants. Passed to kernels by value inside the launch parameters.
struct Cuts {
  float half_kappa_max;
  float z_lum;
  float md_cos_eps[6];
  float md_sin_eps[6];
  float md_dz_res[6];
  float md_eps[6];
  float seg_cos_eps;
  float seg_sin_eps;
  float seg_z0_max[5];
  float t3_kappa_max;
  float t3_chi2rz_max[4];
  float sigma_z2[6];
  float inv_sigma_z2[6];
  float t5_dkappa_max;
  float t5_chi2rz_max[2];
  float t5_chi2xy_max;
  float t5_sigma_xy2_scaled;
  float t5_kappa_max;
  // [P] pixel line segment + outer object; index [0] = pixel triplets, [1] = pixel quintuplets
  float pix_dkappa_max[2];
  float pix_inv_var_xy[6];
  float pix_inv_var_rz[6];
  float pix_chi2xy_max[2];
  float pix_chi2rz_max[2];
};

// SINTHR(r, cosE, sinE) = sin(asin(min(1, r * kappa_max / 2)) + eps)
__device__ __forceinline__ float sin_threshold(const Cuts& c, float r, float cosE, float sinE) {
  float t = r * c.half_kappa_max;
  if (t > 1.0f) t = 1.0f;
  return t * cosE + sqrtf(1.0f - t * t) * sinE;
}

// ---- [M] mini-doublet ------------------------------------------------------
struct MdOut {
  float sinA, cross, dot;
};
// lower = (x, y, z, r) of the side-0 hit, upper likewise for side 1. r = sqrtf(x*x + y*y) was
// derived at load time with that exact expression.
__device__ __forceinline__ bool md_select(const Cuts& c, int layer, const float4& lo, const float4& up, MdOut& o) {
  // no early return (see seg_select): the tests are combined at the end, a NaN fails its `<=`
  const float dx = up.x - lo.x, dy = up.y - lo.y;
  // M1: SINANG(xl, yl, dx, dy)
  const float cross = lo.x * dy - lo.y * dx;
  const float dot = lo.x * dx + lo.y * dy;
  const float n2 = (lo.x * lo.x + lo.y * lo.y) * (dx * dx + dy * dy);
  const float sinA = cross / sqrtf(n2);
  // M2
  const float thr = sin_threshold(c, up.w, c.md_cos_eps[layer], c.md_sin_eps[layer]);
  bool ok = (n2 > 0.0f) & (dot > 0.0f) & (fabsf(sinA) <= thr);
  // M3
  const float dr = up.w - lo.w;
  const float lhs = fabsf((up.z - lo.z) - lo.z * dr / lo.w);
  const float rhs = c.z_lum * fabsf(dr) / lo.w + c.md_dz_res[layer];
  ok = ok & (lo.w > 0.0f) & (lhs <= rhs);
  o.sinA = sinA;
  o.cross = cross;
  o.dot = dot;
  return ok;
}

// ---- [S] segment --------------------------------------------------------
struct SegOut {
  float sinS, z0, cross, dot;
};
// ai / ao = anchor (x, y, z, r) of the inner / outer MD; aux = (ur, sinA) of each.
__device__ __forceinline__ bool seg_select(const Cuts& c, int layer_in, const float4& ai, const float2& auxi,
                                           const float4& ao, const float2& auxo, SegOut& o) {
  // Every value is computed by the SPEC expression; the tests are combined at the end instead of returning early (nine in ten
  // candidates that reach this point pass, and without branches all operands are fetched up front).  A division by zero
  // gives an infinity or a NaN, and a NaN fails its `<=` as the SPEC demands.
  const float dx = ao.x - ai.x, dy = ao.y - ai.y;
  // S2
  const float cross = ai.x * dy - ai.y * dx;
  const float dot = ai.x * dx + ai.y * dy;
  const float n2 = (ai.x * ai.x + ai.y * ai.y) * (dx * dx + dy * dy);
  const float sinS = cross / sqrtf(n2);
  const float thr = sin_threshold(c, ao.w, c.seg_cos_eps, c.seg_sin_eps);
  bool ok = (n2 > 0.0f) & (dot > 0.0f) & (fabsf(sinS) <= thr);
  // S3
  const float dr = ao.w - ai.w;
  const float z0 = ai.z - ai.w * (ao.z - ai.z) / dr;
  ok = ok & (dr > 0.0f) & (fabsf(z0) <= c.seg_z0_max[layer_in]);
  // S4
  const float e1 = fabsf(auxi.y - sinS * (auxi.x / ao.w));
  const float e2 = fabsf(auxo.y - sinS * (auxo.x / ao.w));
  ok = ok & (e1 <= c.md_eps[layer_in]) & (e2 <= c.md_eps[layer_in + 1]);
  o.sinS = sinS;
  o.z0 = z0;
  o.cross = cross;
  o.dot = dot;
  return ok;
}

// ---- [T] triplet ------------------------------------------------------------
__device__ __forceinline__ bool t3_select(const Cuts& c, int layer1, const float4& p1, const float4& p2,
                                          const float4& p3, float& kappa, float& chi2rz) {
  // no early return (see seg_select)
  const float ax = p2.x - p1.x, ay = p2.y - p1.y;
  const float bx = p3.x - p1.x, by = p3.y - p1.y;
  const float cx = p3.x - p2.x, cy = p3.y - p2.y;
  // T2
  const float cross = ax * by - ay * bx;
  const float den2 = ((ax * ax + ay * ay) * (bx * bx + by * by)) * (cx * cx + cy * cy);
  const float k = (2.0f * cross) / sqrtf(den2);
  bool ok = (den2 > 0.0f) & (fabsf(k) <= c.t3_kappa_max);
  // T3
  const float d31 = p3.w - p1.w;
  const float w1 = (p3.w - p2.w) / d31;
  const float w3 = (p2.w - p1.w) / d31;
  const float delta = (p2.z - p1.z) - w3 * (p3.z - p1.z);
  const float var = (c.sigma_z2[layer1 + 1] + (w1 * w1) * c.sigma_z2[layer1]) + (w3 * w3) * c.sigma_z2[layer1 + 2];
  const float chi2 = (delta * delta) / var;
  ok = ok & (d31 > 0.0f) & (chi2 <= c.t3_chi2rz_max[layer1]);
  kappa = k;
  chi2rz = chi2;
  return ok;
}

// ---- [Q] quintuplet ---------------------------------------------------------
struct T5Out {
  float kfit, chi2xy, chi2rz;
};
__device__ __forceinline__ bool t5_select(const Cuts& c, int layer1, float kappaA, float kappaB,
                                          const float4 (&p)[5], T5Out& o) {
  // no early return (see seg_select): the tests are combined at the end
  // Q2
  const float dk = fabsf(kappaA - kappaB);
  bool ok = dk <= c.t5_dkappa_max;
  // Q3: weighted straight line z = a + b r through the five anchors, relative to anchor 2
  float chi2rz;
  {
    float rho[5], zeta[5], w[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
      rho[i] = p[i].w - p[2].w;
      zeta[i] = p[i].z - p[2].z;
      w[i] = c.inv_sigma_z2[layer1 + i];
    }
    float Sw = 0.0f, Sr = 0.0f, Sz = 0.0f, Srr = 0.0f, Srz = 0.0f;
#pragma unroll
    for (int i = 0; i < 5; ++i) {
      Sw = Sw + w[i];
      Sr = Sr + w[i] * rho[i];
      Sz = Sz + w[i] * zeta[i];
      Srr = Srr + (w[i] * rho[i]) * rho[i];
      Srz = Srz + (w[i] * rho[i]) * zeta[i];
    }
    const float D = Sw * Srr - Sr * Sr;
    ok = ok & (D > 0.0f);
    const float b = (Sw * Srz - Sr * Sz) / D;
    const float a = (Sz - b * Sr) / Sw;
    float chi2 = 0.0f;
#pragma unroll
    for (int i = 0; i < 5; ++i) {
      const float e = zeta[i] - (a + b * rho[i]);
      chi2 = chi2 + w[i] * (e * e);
    }
    ok = ok & (chi2 <= c.t5_chi2rz_max[layer1]);
    chi2rz = chi2;
  }
  // Q4: circle fit in the chord frame, lengths scaled by 1/32
  float ex = p[4].x - p[0].x, ey = p[4].y - p[0].y;
  const float len = sqrtf(ex * ex + ey * ey);
  ok = ok & (len > 0.0f);
  ex = ex / len;
  ey = ey / len;
  float u[5], v[5], q[5];
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    const float dx = (p[i].x - p[2].x) * 0.03125f;
    const float dy = (p[i].y - p[2].y) * 0.03125f;
    u[i] = dx * ex + dy * ey;
    v[i] = ex * dy - ey * dx;
    q[i] = u[i] * u[i] + v[i] * v[i];
  }
  float Sqq = 0.0f, Squ = 0.0f, Sq = 0.0f, Suu = 0.0f, Su = 0.0f, Sqv = 0.0f, Suv = 0.0f, Sv = 0.0f;
  const float n = 5.0f;
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    Sqq = Sqq + q[i] * q[i];
    Squ = Squ + q[i] * u[i];
    Sq = Sq + q[i];
    Suu = Suu + u[i] * u[i];
    Su = Su + u[i];
    Sqv = Sqv + q[i] * v[i];
    Suv = Suv + u[i] * v[i];
    Sv = Sv + v[i];
  }
  const float c00 = Suu * n - Su * Su;
  const float c01 = Sq * Su - Squ * n;
  const float c02 = Squ * Su - Sq * Suu;
  const float c11 = Sqq * n - Sq * Sq;
  const float c12 = Squ * Sq - Sqq * Su;
  const float c22 = Sqq * Suu - Squ * Squ;
  const float det = (Sqq * c00 + Squ * c01) + Sq * c02;
  ok = ok & (det > 0.0f);
  const float A = ((c00 * Sqv + c01 * Suv) + c02 * Sv) / det;
  const float B = ((c01 * Sqv + c11 * Suv) + c12 * Sv) / det;
  const float C = ((c02 * Sqv + c12 * Suv) + c22 * Sv) / det;
  float ss = 0.0f;
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    const float e = v[i] - ((A * q[i] + B * u[i]) + C);
    ss = ss + e * e;
  }
  const float chi2xy = ss / c.t5_sigma_xy2_scaled;
  ok = ok & (chi2xy <= c.t5_chi2xy_max);
  // Q5
  const float disc = (1.0f + B * B) - (4.0f * A) * C;
  const float kfit = ((2.0f * A) / sqrtf(disc)) * 0.03125f;
  ok = ok & (disc > 0.0f) & (fabsf(kfit) <= c.t5_kappa_max);
  o.kfit = kfit;
  o.chi2xy = chi2xy;
  o.chi2rz = chi2rz;
  return ok;
}

// ---- [P] pixel line segment + outer object -------------------------------
// "the straight lines and circles in the r-z and x-y plane, respectively, are not fit but rather the estimates from the
// pixel detector are used and the consistency of the outer hits to this hypothesis is checked".
// seed = (kappa, cos phi0, sin phi0, z0, t); the outer object brings N = 3 (triplet, kind 0) or 5 (quintuplet, kind 1)
// anchors on layers layer1 .. layer1 + N - 1 and its own curvature kobj.
struct PixOut {
  float chi2xy, chi2rz, dk;
};
template <int N>
__device__ __forceinline__ bool pix_select(const Cuts& c, int kind, int layer1, float kappa, float cphi, float sphi,
                                           float z0, float t, float kobj, const float4 (&p)[N], PixOut& o) {
  const float hk = 0.5f * kappa;
  // no early return (see seg_select)
  // P0: the first anchor lies ahead of the seed (the outgoing arc of the circle)
  bool ok = p[0].x * cphi + p[0].y * sphi > 0.0f;
  // P1
  const float dk = kobj - kappa;
  ok = ok & (fabsf(dk) <= c.pix_dkappa_max[kind]);
  // P2: distance of the anchors from the seed's circle through the beam line
  float chi2xy = 0.0f;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const float e = (hk * (p[i].w * p[i].w) + p[i].x * sphi) - p[i].y * cphi;
    chi2xy = chi2xy + (e * e) * c.pix_inv_var_xy[layer1 + i];
  }
  ok = ok & (chi2xy <= c.pix_chi2xy_max[kind]);
  // P3: distance of the anchors from the seed's line z = z0 + t s, s = arc length by its power series in (kappa r / 2)^2
  float chi2rz = 0.0f;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const float r = p[i].w;
    const float u = hk * r, u2 = u * u;
    const float s = r * (1.0f + u2 * (0.16666667f + u2 * (0.075f + u2 * (0.04464286f + u2 * (0.030381944f + u2 * 0.022372158f)))));
    const float d = (p[i].z - z0) - t * s;
    chi2rz = chi2rz + (d * d) * c.pix_inv_var_rz[layer1 + i];
  }
  ok = ok & (chi2rz <= c.pix_chi2rz_max[kind]);
  o.chi2xy = chi2xy;
  o.chi2rz = chi2rz;
  o.dk = dk;
  return ok;
}

}  // namespace lst
