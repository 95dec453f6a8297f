/*
 * lst_oracle.c -- ORACLE for the Line Segment Tracking hot path (arXiv 2207.08207).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant generator with the CUDA path (paper_2207_08207_b200/csrc):
 * every constant below is typed here by hand from DESIGN.md section "SPEC".
 *
 * What it is: a plain, slow, single-threaded CPU implementation of
 *     hits -> mini-doublets (MD) -> segments (LS) -> triplets (T3) -> quintuplets (T5)
 * following the paper's order (PAPER.md:37 overview, :43 MD, :47-49 LS + module map,
 * :53 T3, :55 T5).  The paper gives the structure and one number (pT threshold 0.8 GeV,
 * PAPER.md:49); every formula is the reading frozen in DESIGN.md "SPEC" (from SURVEY.md
 * 8(c)), cited as [M1..M3], [S1..S4], [T1..T3], [Q1..Q5] below.  The method is a sequence of
 * cuts, so the result is the SET of objects that pass; no stage picks a "best" candidate.
 *
 * Built twice from this one file:
 *   -DLSTO_F64=0  real = float   the SPEC arithmetic: fp32, round-to-nearest, the exact
 *                                operation order written here, no FMA contraction
 *                                (compile with -ffp-contract=off, no -ffast-math).  This is
 *                                the build GPU parity is checked against.
 *   -DLSTO_F64=1  real = double  same expressions in fp64: used by the CPU tests to pin the
 *                                formulas against closed forms / library fits tightly, and
 *                                to measure how ill-conditioned a quantity is in fp32.
 *
 * Pins (tests/test_oracle_pins.py, tests/test_oracle_events.py): helix closed forms (P1, P2), brute force vs
 * map (P3), single-helix recovery (P4), library least-squares / circumradius reductions (P5),
 * chi2 statistics (P6), symmetries (P7), threshold flips (P8), structure (P9), truth (P10), M3 closed form
 * and flip (P18), per-layer threshold indices (P19), the Q5 cut (P20);
 * duplicate cleaning [D] (tests/test_oracle_clean.py): single helix (P11), set-based restatement (P12),
 * implied properties and order independence (P13), truth statistics (P14); module-map builder [B]
 * (tests/test_oracle_map.py): simulated tracks stay inside the map (P15), the test-side generator (P16: a
 * restatement, pins nothing on its own), symmetries and monotonicity (P17), two-module special cases by
 * similar triangles / arc lengths (P18), helices propagated from the module edges: soundness and tightness (P19).
 * Every pin was checked to bite by mutating this file (a dropped term, a wrong index, a removed cut).
 * The paper prints no worked numerical example, so no value is pinned to the paper itself.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef LSTO_F64
#define LSTO_F64 0
#endif
#if LSTO_F64
typedef double real;
#define R_SQRT sqrt
#define R_ABS fabs
#define R_ATAN2 atan2
#define C(x) x
#else
typedef float real;
#define R_SQRT sqrtf
#define R_ABS fabsf
#define R_ATAN2 atan2f
#define C(x) x##f
#endif

#define N_LAYERS 6

/* ------------------------------------------------------------------------------------ */
/* Cut constants (DESIGN.md "SPEC" table). cm, GeV, tesla, radians.                       */
/* ------------------------------------------------------------------------------------ */
typedef struct {
  real half_kappa_max;          /* 0.5 * k*B/PT_MIN, k = 2.99792458e-3, B = 3.8, PT_MIN = 0.8 */
  real z_lum;                   /* luminous region half-length (3 sigma of the generator)     */
  real md_cos_eps[N_LAYERS];    /* cos / sin of EPS_MD[l] = 4*sqrt(2)*sigma_rphi/gap[l]       */
  real md_sin_eps[N_LAYERS];
  real md_dz_res[N_LAYERS];     /* 4*sqrt(2)*sigma_z[l]                                       */
  real md_eps[N_LAYERS];        /* EPS_MD[l] in sine units, used by S4                        */
  real seg_cos_eps, seg_sin_eps;/* cos / sin of EPS_SEG = 0.002                               */
  real seg_z0_max[N_LAYERS-1];  /* ZSEG by inner layer                                        */
  real t3_kappa_max;            /* 1.05 * KAPPA_MAX                                           */
  real t3_chi2rz_max[N_LAYERS-2];
  real sigma_z2[N_LAYERS];      /* sigma_z[l]^2                                               */
  real inv_sigma_z2[N_LAYERS];  /* 1/sigma_z[l]^2                                             */
  real t5_dkappa_max;           /* 0.02 * KAPPA_MAX                                           */
  real t5_chi2rz_max[N_LAYERS-4];
  real t5_chi2xy_max;
  real t5_sigma_xy2_scaled;     /* (sigma_rphi/32)^2                                          */
  real t5_kappa_max;            /* 1.05 * KAPPA_MAX                                           */
  /* [P] pixel line segments -> pT3 / pT5; index [0] = pixel triplets, [1] = pixel quintuplets */
  real pix_dkappa_max[2];       /* |kappa of the outer object - kappa of the seed|            */
  real pix_inv_var_xy[N_LAYERS];/* 1 / (x-y variance of an anchor of layer l about the seed's circle) */
  real pix_inv_var_rz[N_LAYERS];/* 1 / (z variance of an anchor of layer l about the seed's line)     */
  real pix_chi2xy_max[2];
  real pix_chi2rz_max[2];
} lsto_config;

void lsto_default_config(lsto_config* c) {
  int l;
  c->half_kappa_max = C(0.00712007098);
  c->z_lum = C(15.0);
  for (l = 0; l < N_LAYERS; ++l) {
    int ps = l < 3;
    c->md_cos_eps[l] = ps ? C(0.99840045) : C(0.995777965);
    c->md_sin_eps[l] = ps ? C(0.056538377) : C(0.0917944759);
    c->md_dz_res[l]  = ps ? C(0.243244737) : C(7.91959572);
    c->md_eps[l]     = ps ? C(0.0565685406) : C(0.091923885);
    c->sigma_z2[l]     = ps ? C(0.001849) : C(1.96);
    c->inv_sigma_z2[l] = ps ? C(540.832886) : C(0.510204077);
  }
  c->seg_cos_eps = C(0.999997973);
  c->seg_sin_eps = C(0.0019999987);
  c->seg_z0_max[0] = C(20.0); c->seg_z0_max[1] = C(20.0); c->seg_z0_max[2] = C(40.0);
  c->seg_z0_max[3] = C(90.0); c->seg_z0_max[4] = C(90.0);
  c->t3_kappa_max = C(0.0149521492);
  c->t3_chi2rz_max[0] = C(100.0); c->t3_chi2rz_max[1] = C(30.0);
  c->t3_chi2rz_max[2] = C(25.0);  c->t3_chi2rz_max[3] = C(25.0);
  c->t5_dkappa_max = C(0.000284802838);
  c->t5_chi2rz_max[0] = C(110.0); c->t5_chi2rz_max[1] = C(150.0);
  c->t5_chi2xy_max = C(35.0);
  c->t5_sigma_xy2_scaled = C(6.6015625e-09);
  c->t5_kappa_max = C(0.0149521492);
  c->pix_dkappa_max[0] = C(0.0008); c->pix_dkappa_max[1] = C(0.0007);
  c->pix_inv_var_xy[0] = C(809.479);   c->pix_inv_var_xy[1] = C(187.19363); c->pix_inv_var_xy[2] = C(51.984085);
  c->pix_inv_var_xy[3] = C(16.645065); c->pix_inv_var_xy[4] = C(6.149085);  c->pix_inv_var_xy[5] = C(2.8425808);
  c->pix_inv_var_rz[0] = C(229.09508);  c->pix_inv_var_rz[1] = C(136.11072); c->pix_inv_var_rz[2] = C(79.544624);
  c->pix_inv_var_rz[3] = C(0.50524855); c->pix_inv_var_rz[4] = C(0.5020406); c->pix_inv_var_rz[5] = C(0.4982422);
  c->pix_chi2xy_max[0] = C(85.0); c->pix_chi2xy_max[1] = C(145.0);
  c->pix_chi2rz_max[0] = C(25.0); c->pix_chi2rz_max[1] = C(35.0);
}

int lsto_is_f64(void) { return LSTO_F64; }
int lsto_sizeof_config(void) { return (int)sizeof(lsto_config); }

/* ------------------------------------------------------------------------------------ */
/* Helpers shared by the cuts (SINANG, SINTHR)                          */
/* ------------------------------------------------------------------------------------ */

/* Sine of the angle from the position vector p=(px,py) to the direction d=(dx,dy), and
 * their dot product. Returns 0 (reject) if either vector has zero length. */
static int sinang(real px, real py, real dx, real dy, real* sinA, real* cross, real* dot) {
  real n2;
  *cross = px * dy - py * dx;
  *dot = px * dx + py * dy;
  n2 = (px * px + py * py) * (dx * dx + dy * dy);
  if (!(n2 > C(0.0))) return 0;
  *sinA = *cross / R_SQRT(n2);
  return 1;
}

/* sin(asin(t) + eps) with t = min(1, r * kappa_max/2): the largest |sinA| a particle from the
 * beam line with pT >= PT_MIN can show at radius r, widened by the angle eps. */
static real sinthr(const lsto_config* c, real r, real cosE, real sinE) {
  real t = r * c->half_kappa_max;
  if (t > C(1.0)) t = C(1.0);
  return t * cosE + R_SQRT(C(1.0) - t * t) * sinE;
}

/* ------------------------------------------------------------------------------------ */
/* [M] mini-doublet: one hit on each sensor of one module                   */
/* out[0]=sinA out[1]=dphi out[2]=dphichange out[3]=r_l out[4]=r_u                         */
/* margin[k] = {value, threshold} pairs of M2, M3 (filled as far as evaluated)            */
/* ------------------------------------------------------------------------------------ */
int lsto_md_cut(const lsto_config* c, int layer,
                real xl, real yl, real zl, real xu, real yu, real zu,
                real* out, real* margin) {
  real rl = R_SQRT(xl * xl + yl * yl);
  real ru = R_SQRT(xu * xu + yu * yu);
  real dx = xu - xl, dy = yu - yl;
  real sinA, cross, dot, thr, dr, lhs, rhs;
  /* M1: slope of the hit pair relative to the radial direction at the lower hit */
  if (!sinang(xl, yl, dx, dy, &sinA, &cross, &dot)) return 0;
  if (!(dot > C(0.0))) return 0;
  /* M2: consistent with pT >= PT_MIN for a particle from the beam line, + resolution term */
  thr = sinthr(c, ru, c->md_cos_eps[layer], c->md_sin_eps[layer]);
  if (margin) { margin[0] = R_ABS(sinA); margin[1] = thr; }
  if (!(R_ABS(sinA) <= thr)) return 0;
  /* M3: z compatibility with a straight line from the luminous region in r-z */
  if (!(rl > C(0.0))) return 0;
  dr = ru - rl;
  lhs = R_ABS((zu - zl) - zl * dr / rl);
  rhs = c->z_lum * R_ABS(dr) / rl + c->md_dz_res[layer];
  if (margin) { margin[2] = lhs; margin[3] = rhs; }
  if (!(lhs <= rhs)) return 0;
  out[0] = sinA;
  out[1] = R_ATAN2(xl * yu - yl * xu, xl * xu + yl * yu);
  out[2] = R_ATAN2(cross, dot);
  out[3] = rl;
  out[4] = ru;
  return 1;
}

/* ------------------------------------------------------------------------------------ */
/* [S] segment: two MDs on map-connected modules of adjacent layers      */
/* inner MD: anchor (xi,yi,zi,ri), upper-hit radius uri, sinAi; outer likewise.            */
/* out[0]=sinS out[1]=z0 out[2]=dphi out[3]=dphichange                                     */
/* ------------------------------------------------------------------------------------ */
int lsto_seg_cut(const lsto_config* c, int layer_in,
                 real xi, real yi, real zi, real ri, real uri, real sinAi,
                 real xo, real yo, real zo, real ro, real uro, real sinAo,
                 real* out, real* margin) {
  real dx = xo - xi, dy = yo - yi;
  real sinS, cross, dot, thr, dr, z0, e1, e2;
  /* S2: pT of the anchor-to-anchor direction */
  if (!sinang(xi, yi, dx, dy, &sinS, &cross, &dot)) return 0;
  if (!(dot > C(0.0))) return 0;
  thr = sinthr(c, ro, c->seg_cos_eps, c->seg_sin_eps);
  if (margin) { margin[0] = R_ABS(sinS); margin[1] = thr; }
  if (!(R_ABS(sinS) <= thr)) return 0;
  /* S3: straight line in r-z points back to the luminous region */
  dr = ro - ri;
  if (!(dr > C(0.0))) return 0;
  z0 = zi - ri * (zo - zi) / dr;
  if (margin) { margin[2] = R_ABS(z0); margin[3] = c->seg_z0_max[layer_in]; }
  if (!(R_ABS(z0) <= c->seg_z0_max[layer_in])) return 0;
  /* S4: each MD's own slope agrees with the segment's circle through the beam line
   * (sin(alpha) is proportional to r on such a circle) */
  e1 = R_ABS(sinAi - sinS * (uri / ro));
  if (margin) { margin[4] = e1; margin[5] = c->md_eps[layer_in]; }
  if (!(e1 <= c->md_eps[layer_in])) return 0;
  e2 = R_ABS(sinAo - sinS * (uro / ro));
  if (margin) { margin[6] = e2; margin[7] = c->md_eps[layer_in + 1]; }
  if (!(e2 <= c->md_eps[layer_in + 1])) return 0;
  out[0] = sinS;
  out[1] = z0;
  out[2] = R_ATAN2(xi * yo - yi * xo, xi * xo + yi * yo);
  out[3] = R_ATAN2(cross, dot);
  return 1;
}

/* ------------------------------------------------------------------------------------ */
/* [T] triplet: two segments sharing an MD; anchors p1,p2,p3 on layers l, l+1, l+2         */
/* (PAPER.md:53). p = {x,y,z,r}.  out[0]=kappa out[1]=chi2rz                               */
/* ------------------------------------------------------------------------------------ */
int lsto_t3_cut(const lsto_config* c, int layer1,
                const real* p1, const real* p2, const real* p3, real* out, real* margin) {
  real ax = p2[0] - p1[0], ay = p2[1] - p1[1];
  real bx = p3[0] - p1[0], by = p3[1] - p1[1];
  real cx = p3[0] - p2[0], cy = p3[1] - p2[1];
  real cross, den2, kappa, d31, w1, w3, delta, var, chi2;
  /* T2: signed curvature of the circle through the three anchors ("trivially created
   * from the three points"): 2*cross / (|a||b||c|) */
  cross = ax * by - ay * bx;
  den2 = ((ax * ax + ay * ay) * (bx * bx + by * by)) * (cx * cx + cy * cy);
  if (!(den2 > C(0.0))) return 0;
  kappa = (C(2.0) * cross) / R_SQRT(den2);
  if (margin) { margin[0] = R_ABS(kappa); margin[1] = c->t3_kappa_max; }
  if (!(R_ABS(kappa) <= c->t3_kappa_max)) return 0;
  /* T3: chi2 of a straight line through the three anchors in r-z (1 dof, closed form):
   * residual of the middle anchor from the chord of the outer two */
  d31 = p3[3] - p1[3];
  if (!(d31 > C(0.0))) return 0;
  w1 = (p3[3] - p2[3]) / d31;
  w3 = (p2[3] - p1[3]) / d31;
  delta = (p2[2] - p1[2]) - w3 * (p3[2] - p1[2]);
  var = (c->sigma_z2[layer1 + 1] + (w1 * w1) * c->sigma_z2[layer1]) + (w3 * w3) * c->sigma_z2[layer1 + 2];
  chi2 = (delta * delta) / var;
  if (margin) { margin[2] = chi2; margin[3] = c->t3_chi2rz_max[layer1]; }
  if (!(chi2 <= c->t3_chi2rz_max[layer1])) return 0;
  out[0] = kappa;
  out[1] = chi2;
  return 1;
}

/* ------------------------------------------------------------------------------------ */
/* [Q] quintuplet: two triplets sharing an MD; anchors p[0..4] on layers l..l+4            */
/* (PAPER.md:55). out[0]=kFit out[1]=chi2xy out[2]=chi2rz                                  */
/* ------------------------------------------------------------------------------------ */
int lsto_t5_cut(const lsto_config* c, int layer1, real kappaA, real kappaB,
                const real* p /* [5][4] x,y,z,r */, real* out, real* margin) {
  int i;
  real dk;
  /* Q2: circles of the inner and outer triplet have "radii close to each other":
   * compared as signed curvatures (radii are unbounded for straight tracks) */
  dk = R_ABS(kappaA - kappaB);
  if (margin) { margin[0] = dk; margin[1] = c->t5_dkappa_max; }
  if (!(dk <= c->t5_dkappa_max)) return 0;

  /* Q3: weighted least-squares straight line z = a + b*r through the five anchors,
   * weights 1/sigma_z^2, coordinates taken relative to the middle anchor */
  {
    real rho[5], zeta[5], w[5];
    real Sw = C(0.0), Sr = C(0.0), Sz = C(0.0), Srr = C(0.0), Srz = C(0.0);
    real D, a, b, chi2 = C(0.0);
    for (i = 0; i < 5; ++i) {
      rho[i] = p[4 * i + 3] - p[4 * 2 + 3];
      zeta[i] = p[4 * i + 2] - p[4 * 2 + 2];
      w[i] = c->inv_sigma_z2[layer1 + i];
    }
    for (i = 0; i < 5; ++i) {
      Sw = Sw + w[i];
      Sr = Sr + w[i] * rho[i];
      Sz = Sz + w[i] * zeta[i];
      Srr = Srr + (w[i] * rho[i]) * rho[i];
      Srz = Srz + (w[i] * rho[i]) * zeta[i];
    }
    D = Sw * Srr - Sr * Sr;
    if (!(D > C(0.0))) return 0;
    b = (Sw * Srz - Sr * Sz) / D;
    a = (Sz - b * Sr) / Sw;
    for (i = 0; i < 5; ++i) {
      real e = zeta[i] - (a + b * rho[i]);
      chi2 = chi2 + w[i] * (e * e);
    }
    if (margin) { margin[2] = chi2; margin[3] = c->t5_chi2rz_max[layer1]; }
    if (!(chi2 <= c->t5_chi2rz_max[layer1])) return 0;
    out[2] = chi2;
  }

  /* Q4: global circle fit of the five anchors in x-y. Frame: origin at the middle anchor,
   * u along the chord p1->p5, v to its left, lengths scaled by 1/32 (exact). A circle obeys
   * v = A*(u^2+v^2) + B*u + C exactly; least squares over (A,B,C), 3x3 normal equations by
   * cofactors in a fixed order; chi2 = sum of squared v-residuals / sigma_rphi^2. */
  {
    real ex = p[4 * 4 + 0] - p[0], ey = p[4 * 4 + 1] - p[1];
    real L = R_SQRT(ex * ex + ey * ey);
    real u[5], v[5], q[5];
    real Sqq = C(0.0), Squ = C(0.0), Sq = C(0.0), Suu = C(0.0), Su = C(0.0);
    real Sqv = C(0.0), Suv = C(0.0), Sv = C(0.0), n = C(5.0);
    real c00, c01, c02, c11, c12, c22, det, A, B, Cc, ss = C(0.0), chi2, disc, kfit;
    if (!(L > C(0.0))) return 0;
    ex = ex / L; ey = ey / L;
    for (i = 0; i < 5; ++i) {
      real dx = (p[4 * i + 0] - p[4 * 2 + 0]) * C(0.03125);
      real dy = (p[4 * i + 1] - p[4 * 2 + 1]) * C(0.03125);
      u[i] = dx * ex + dy * ey;
      v[i] = ex * dy - ey * dx;
      q[i] = u[i] * u[i] + v[i] * v[i];
    }
    for (i = 0; i < 5; ++i) {
      Sqq = Sqq + q[i] * q[i];
      Squ = Squ + q[i] * u[i];
      Sq = Sq + q[i];
      Suu = Suu + u[i] * u[i];
      Su = Su + u[i];
      Sqv = Sqv + q[i] * v[i];
      Suv = Suv + u[i] * v[i];
      Sv = Sv + v[i];
    }
    /* M = [[Sqq Squ Sq],[Squ Suu Su],[Sq Su n]], rhs = (Sqv, Suv, Sv) */
    c00 = Suu * n - Su * Su;
    c01 = Sq * Su - Squ * n;
    c02 = Squ * Su - Sq * Suu;
    c11 = Sqq * n - Sq * Sq;
    c12 = Squ * Sq - Sqq * Su;
    c22 = Sqq * Suu - Squ * Squ;
    det = (Sqq * c00 + Squ * c01) + Sq * c02;
    if (!(det > C(0.0))) return 0;
    A = ((c00 * Sqv + c01 * Suv) + c02 * Sv) / det;
    B = ((c01 * Sqv + c11 * Suv) + c12 * Sv) / det;
    Cc = ((c02 * Sqv + c12 * Suv) + c22 * Sv) / det;
    for (i = 0; i < 5; ++i) {
      real e = v[i] - ((A * q[i] + B * u[i]) + Cc);
      ss = ss + e * e;
    }
    chi2 = ss / c->t5_sigma_xy2_scaled;
    if (margin) { margin[4] = chi2; margin[5] = c->t5_chi2xy_max; }
    if (!(chi2 <= c->t5_chi2xy_max)) return 0;
    /* Q5: curvature of the fitted circle, back in cm^-1 */
    disc = (C(1.0) + B * B) - (C(4.0) * A) * Cc;
    if (!(disc > C(0.0))) return 0;
    kfit = ((C(2.0) * A) / R_SQRT(disc)) * C(0.03125);
    if (margin) { margin[6] = R_ABS(kfit); margin[7] = c->t5_kappa_max; }
    if (!(R_ABS(kfit) <= c->t5_kappa_max)) return 0;
    out[0] = kfit;
    out[1] = chi2;
  }
  return 1;
}

/* ------------------------------------------------------------------------------------ */
/* [P] pixel line segment + outer object -> pixel triplet / pixel quintuplet */
/* ------------------------------------------------------------------------------------ */
/* "Selections similar to that used for the Quintuplets are used here, the difference being that the straight lines
 * and circles in the r-z and x-y plane, respectively, are not fit but rather the estimates from the pixel detector
 * are used and the consistency of the outer hits to this hypothesis is checked".  Reading (DESIGN.md
 * SPEC [P], reading 28): a pixel line segment is the inner tracker's estimate of a prompt helix,
 *     seed = (kappa, cos phi0, sin phi0, z0, t):  signed curvature (sign as the triplet's kappa), direction of the
 *     momentum at the beam line, z at the beam line, t = cot(theta) = dz / d(arc length);
 * the outer object brings n = 3 (triplet) or 5 (quintuplet) anchors p_i on layers layer1 .. layer1 + n - 1 and its own
 * curvature kappa_obj (circumcurvature of the triplet / fitted curvature of the quintuplet).
 *   P0  the first anchor lies ahead of the seed: x_1 cos phi0 + y_1 sin phi0 > 0 (a circle through the beam line passes
 *       every radius twice, going out and coming back; e(p) below vanishes on both arcs, the outer tracker's hits of a
 *       prompt particle sit on the outgoing one)
 *   P1  |kappa_obj - kappa| <= pix_dkappa_max[kind]                  ("radii close to each other", with the seed's)
 *   P2  x-y: the seed's circle goes through the beam line with that direction and curvature; a point p lies on it iff
 *       e(p) = (kappa / 2) r^2 + x sin phi0 - y cos phi0 = 0, and e is the signed distance from the circle to first
 *       order (its gradient has unit length on the circle).  chi2xy = sum_i e_i^2 / var_xy[layer_i] <= pix_chi2xy_max[kind]
 *   P3  r-z: the seed's line is z = z0 + t s, s the arc length in the transverse plane at radius r,
 *       s = (2 / kappa) asin(kappa r / 2), taken by its power series in u^2 = (kappa r / 2)^2 up to u^10 (no
 *       transcendental function in a cut variable; remainder < 0.035 u^12 r for u <= 0.77, the largest value in this geometry).  d_i = (z_i - z0) - t s_i;
 *       chi2rz = sum_i d_i^2 / var_rz[layer_i] <= pix_chi2rz_max[kind]
 * kind: 0 = pixel triplet, 1 = pixel quintuplet.  p = [n][4] x, y, z, r.
 * out[0] = chi2xy, out[1] = chi2rz, out[2] = kappa_obj - kappa; margin = {value, threshold} of P1, P2, P3. */
int lsto_pix_cut(const lsto_config* c, int kind, int layer1, int n, const real* seed /* kappa, cphi, sphi, z0, t */,
                 real kappa_obj, const real* p, real* out, real* margin) {
  const real kappa = seed[0], cphi = seed[1], sphi = seed[2], z0 = seed[3], t = seed[4];
  const real hk = C(0.5) * kappa;
  real dk, chi2xy = C(0.0), chi2rz = C(0.0);
  int i;
  /* P0 */
  if (!(p[0] * cphi + p[1] * sphi > C(0.0))) return 0;
  /* P1 */
  dk = kappa_obj - kappa;
  if (margin) { margin[0] = R_ABS(dk); margin[1] = c->pix_dkappa_max[kind]; }
  if (!(R_ABS(dk) <= c->pix_dkappa_max[kind])) return 0;
  /* P2 */
  for (i = 0; i < n; ++i) {
    const real x = p[4 * i + 0], y = p[4 * i + 1], r = p[4 * i + 3];
    const real e = (hk * (r * r) + x * sphi) - y * cphi;
    chi2xy = chi2xy + (e * e) * c->pix_inv_var_xy[layer1 + i];
  }
  if (margin) { margin[2] = chi2xy; margin[3] = c->pix_chi2xy_max[kind]; }
  if (!(chi2xy <= c->pix_chi2xy_max[kind])) return 0;
  /* P3 */
  for (i = 0; i < n; ++i) {
    const real z = p[4 * i + 2], r = p[4 * i + 3];
    const real u = hk * r, u2 = u * u;
    const real s = r * (C(1.0) + u2 * (C(0.16666667) + u2 * (C(0.075) + u2 * (C(0.04464286) + u2 * (C(0.030381944) + u2 * C(0.022372158))))));
    const real d = (z - z0) - t * s;
    chi2rz = chi2rz + (d * d) * c->pix_inv_var_rz[layer1 + i];
  }
  if (margin) { margin[4] = chi2rz; margin[5] = c->pix_chi2rz_max[kind]; }
  if (!(chi2rz <= c->pix_chi2rz_max[kind])) return 0;
  out[0] = chi2xy;
  out[1] = chi2rz;
  out[2] = dk;
  return 1;
}

/* ------------------------------------------------------------------------------------ */
/* Event-level driver                                                                      */
/* ------------------------------------------------------------------------------------ */
typedef struct {
  /* MDs */
  int64_t n_md, cap_md;
  int32_t *md_lower, *md_upper, *md_module;          /* original hit indices, module id      */
  real *md_x, *md_y, *md_z, *md_r, *md_ur, *md_sinA, *md_dphi, *md_dphichange;
  /* segments */
  int64_t n_seg, cap_seg;
  int32_t *seg_in, *seg_out;                         /* MD indices                            */
  real *seg_sinS, *seg_z0, *seg_dphi, *seg_dphichange;
  /* triplets */
  int64_t n_t3, cap_t3;
  int32_t *t3_a, *t3_b;                              /* segment indices                       */
  real *t3_kappa, *t3_chi2rz;
  /* quintuplets */
  int64_t n_t5, cap_t5;
  int32_t *t5_a, *t5_b;                              /* triplet indices                       */
  real *t5_kfit, *t5_chi2xy, *t5_chi2rz;
  /* candidates examined per stage */
  int64_t cand[4];
  /* [P] pixel links of kind 0 (pT3) / 1 (pT5): seed index, index of the outer object, chi2xy, chi2rz, kappa_obj - kappa */
  int64_t n_pix[2], cap_pix[2], cand_pix[2];
  int32_t *pix_seed[2], *pix_obj[2];
  real *pix_chi2xy[2], *pix_chi2rz[2], *pix_dk[2];
} lsto_event;

static void* grow(void* p, int64_t n, size_t sz) { return realloc(p, (size_t)(n > 0 ? n : 1) * sz); }

#define GROW_MD(ev)  do { if ((ev)->n_md == (ev)->cap_md) { int64_t c = (ev)->cap_md ? 2*(ev)->cap_md : 1024; \
  (ev)->md_lower = grow((ev)->md_lower, c, 4); (ev)->md_upper = grow((ev)->md_upper, c, 4); \
  (ev)->md_module = grow((ev)->md_module, c, 4); \
  (ev)->md_x = grow((ev)->md_x, c, sizeof(real)); (ev)->md_y = grow((ev)->md_y, c, sizeof(real)); \
  (ev)->md_z = grow((ev)->md_z, c, sizeof(real)); (ev)->md_r = grow((ev)->md_r, c, sizeof(real)); \
  (ev)->md_ur = grow((ev)->md_ur, c, sizeof(real)); (ev)->md_sinA = grow((ev)->md_sinA, c, sizeof(real)); \
  (ev)->md_dphi = grow((ev)->md_dphi, c, sizeof(real)); (ev)->md_dphichange = grow((ev)->md_dphichange, c, sizeof(real)); \
  (ev)->cap_md = c; } } while (0)
#define GROW_SEG(ev) do { if ((ev)->n_seg == (ev)->cap_seg) { int64_t c = (ev)->cap_seg ? 2*(ev)->cap_seg : 1024; \
  (ev)->seg_in = grow((ev)->seg_in, c, 4); (ev)->seg_out = grow((ev)->seg_out, c, 4); \
  (ev)->seg_sinS = grow((ev)->seg_sinS, c, sizeof(real)); (ev)->seg_z0 = grow((ev)->seg_z0, c, sizeof(real)); \
  (ev)->seg_dphi = grow((ev)->seg_dphi, c, sizeof(real)); (ev)->seg_dphichange = grow((ev)->seg_dphichange, c, sizeof(real)); \
  (ev)->cap_seg = c; } } while (0)
#define GROW_T3(ev)  do { if ((ev)->n_t3 == (ev)->cap_t3) { int64_t c = (ev)->cap_t3 ? 2*(ev)->cap_t3 : 1024; \
  (ev)->t3_a = grow((ev)->t3_a, c, 4); (ev)->t3_b = grow((ev)->t3_b, c, 4); \
  (ev)->t3_kappa = grow((ev)->t3_kappa, c, sizeof(real)); (ev)->t3_chi2rz = grow((ev)->t3_chi2rz, c, sizeof(real)); \
  (ev)->cap_t3 = c; } } while (0)
#define GROW_T5(ev)  do { if ((ev)->n_t5 == (ev)->cap_t5) { int64_t c = (ev)->cap_t5 ? 2*(ev)->cap_t5 : 1024; \
  (ev)->t5_a = grow((ev)->t5_a, c, 4); (ev)->t5_b = grow((ev)->t5_b, c, 4); \
  (ev)->t5_kfit = grow((ev)->t5_kfit, c, sizeof(real)); (ev)->t5_chi2xy = grow((ev)->t5_chi2xy, c, sizeof(real)); \
  (ev)->t5_chi2rz = grow((ev)->t5_chi2rz, c, sizeof(real)); \
  (ev)->cap_t5 = c; } } while (0)

void lsto_free(lsto_event* ev) {
  if (!ev) return;
  free(ev->md_lower); free(ev->md_upper); free(ev->md_module);
  free(ev->md_x); free(ev->md_y); free(ev->md_z); free(ev->md_r); free(ev->md_ur);
  free(ev->md_sinA); free(ev->md_dphi); free(ev->md_dphichange);
  free(ev->seg_in); free(ev->seg_out); free(ev->seg_sinS); free(ev->seg_z0);
  free(ev->seg_dphi); free(ev->seg_dphichange);
  free(ev->t3_a); free(ev->t3_b); free(ev->t3_kappa); free(ev->t3_chi2rz);
  free(ev->t5_a); free(ev->t5_b); free(ev->t5_kfit); free(ev->t5_chi2xy); free(ev->t5_chi2rz);
  { int k; for (k = 0; k < 2; ++k) { free(ev->pix_seed[k]); free(ev->pix_obj[k]); free(ev->pix_chi2xy[k]); free(ev->pix_chi2rz[k]); free(ev->pix_dk[k]); } }
  free(ev);
}

/* Try one segment candidate (MD i, MD o); append if it passes. */
static void try_segment(const lsto_config* cfg, const int8_t* layer, lsto_event* ev, int32_t i, int32_t o) {
  real out[4];
  ev->cand[1]++;
  if (lsto_seg_cut(cfg, layer[ev->md_module[i]],
                   ev->md_x[i], ev->md_y[i], ev->md_z[i], ev->md_r[i], ev->md_ur[i], ev->md_sinA[i],
                   ev->md_x[o], ev->md_y[o], ev->md_z[o], ev->md_r[o], ev->md_ur[o], ev->md_sinA[o],
                   out, NULL)) {
    GROW_SEG(ev);
    ev->seg_in[ev->n_seg] = i; ev->seg_out[ev->n_seg] = o;
    ev->seg_sinS[ev->n_seg] = out[0]; ev->seg_z0[ev->n_seg] = out[1];
    ev->seg_dphi[ev->n_seg] = out[2]; ev->seg_dphichange[ev->n_seg] = out[3];
    ev->n_seg++;
  }
}

/* mode 0: module-driven search over the module map (the method)
 * mode 1: brute force over ALL MD pairs of adjacent layers, kept only if the module pair is
 *         in the map (pin P3(i): must give the same set as mode 0)
 * mode 2: brute force over ALL MD pairs of adjacent layers, map ignored (pin P3(ii))
 * stages: build up to 1 = MD, 2 = LS, 3 = T3, 4 = T5
 * Returns NULL on invalid input (module id / side out of range, bad map). */
lsto_event* lsto_run(const lsto_config* cfg, int32_t n_modules, const int8_t* layer,
                     const int32_t* row_offsets, const int32_t* targets,
                     int32_t n_hits, const float* x, const float* y, const float* z,
                     const int32_t* module, const uint8_t* side, int mode, int stages) {
  lsto_event* ev;
  int32_t *start, *fill, *order, m, h;
  int64_t s, a;
  for (h = 0; h < n_hits; ++h)
    if (module[h] < 0 || module[h] >= n_modules || side[h] > 1) return NULL;
  for (m = 0; m < n_modules; ++m) {
    int32_t k;
    if (layer[m] < 0 || layer[m] >= N_LAYERS || row_offsets[m + 1] < row_offsets[m]) return NULL;
    for (k = row_offsets[m]; k < row_offsets[m + 1]; ++k)
      if (targets[k] < 0 || targets[k] >= n_modules || layer[targets[k]] != layer[m] + 1) return NULL;
  }
  ev = calloc(1, sizeof(*ev));

  /* hits of each (module, side) in input order */
  start = calloc((size_t)2 * n_modules + 1, 4);
  fill = calloc((size_t)2 * n_modules + 1, 4);
  order = malloc((size_t)(n_hits > 0 ? n_hits : 1) * 4);
  for (h = 0; h < n_hits; ++h) start[2 * module[h] + side[h] + 1]++;
  for (m = 0; m < 2 * n_modules; ++m) start[m + 1] += start[m];
  for (h = 0; h < n_hits; ++h) { int32_t b = 2 * module[h] + side[h]; order[start[b] + fill[b]++] = h; }

  /* ---- mini-doublets: every (lower, upper) hit pair of every module ---- */
  for (m = 0; m < n_modules; ++m) {
    int32_t il, iu;
    for (il = start[2 * m]; il < start[2 * m + 1]; ++il)
      for (iu = start[2 * m + 1]; iu < start[2 * m + 2]; ++iu) {
        int32_t l = order[il], u = order[iu];
        real out[5];
        ev->cand[0]++;
        if (lsto_md_cut(cfg, layer[m], x[l], y[l], z[l], x[u], y[u], z[u], out, NULL)) {
          GROW_MD(ev);
          ev->md_lower[ev->n_md] = l; ev->md_upper[ev->n_md] = u; ev->md_module[ev->n_md] = m;
          /* anchor = lower-sensor hit (pixel side on PS, lower side on 2S) */
          ev->md_x[ev->n_md] = x[l]; ev->md_y[ev->n_md] = y[l]; ev->md_z[ev->n_md] = z[l];
          ev->md_r[ev->n_md] = out[3]; ev->md_ur[ev->n_md] = out[4];
          ev->md_sinA[ev->n_md] = out[0]; ev->md_dphi[ev->n_md] = out[1]; ev->md_dphichange[ev->n_md] = out[2];
          ev->n_md++;
        }
      }
  }
  free(fill); free(order);
  if (stages < 2) { free(start); return ev; }

  /* ---- segments ---- */
  {
    /* MDs were appended module by module: mdStart[m] .. mdStart[m+1] */
    int32_t* mdStart = calloc((size_t)n_modules + 1, 4);
    int64_t i, o;
    for (i = 0; i < ev->n_md; ++i) mdStart[ev->md_module[i] + 1]++;
    for (m = 0; m < n_modules; ++m) mdStart[m + 1] += mdStart[m];
    if (mode == 0) {
      for (m = 0; m < n_modules; ++m) {
        int32_t k;
        for (k = row_offsets[m]; k < row_offsets[m + 1]; ++k) {
          int32_t b = targets[k];
          for (i = mdStart[m]; i < mdStart[m + 1]; ++i)
            for (o = mdStart[b]; o < mdStart[b + 1]; ++o)
              try_segment(cfg, layer, ev, (int32_t)i, (int32_t)o);
        }
      }
    } else {
      for (i = 0; i < ev->n_md; ++i)
        for (o = 0; o < ev->n_md; ++o) {
          int32_t ma = ev->md_module[i], mb = ev->md_module[o];
          if (layer[mb] != layer[ma] + 1) continue;
          if (mode == 1) {
            int32_t k, found = 0;
            for (k = row_offsets[ma]; k < row_offsets[ma + 1]; ++k) if (targets[k] == mb) { found = 1; break; }
            if (!found) continue;
          }
          try_segment(cfg, layer, ev, (int32_t)i, (int32_t)o);
        }
    }
    free(mdStart);
  }
  free(start);
  if (stages < 3) return ev;

  /* ---- triplets: segment pairs (a, b) with outer(a) == inner(b) ---- */
  {
    int32_t* byIn = calloc((size_t)ev->n_md + 1, 4);     /* segments grouped by inner MD */
    int32_t* lst = malloc((size_t)(ev->n_seg > 0 ? ev->n_seg : 1) * 4);
    int32_t* cur = calloc((size_t)ev->n_md + 1, 4);
    for (s = 0; s < ev->n_seg; ++s) byIn[ev->seg_in[s] + 1]++;
    for (a = 0; a < ev->n_md; ++a) byIn[a + 1] += byIn[a];
    for (s = 0; s < ev->n_seg; ++s) { int32_t i = ev->seg_in[s]; lst[byIn[i] + cur[i]++] = (int32_t)s; }
    for (a = 0; a < ev->n_seg; ++a) {
      int32_t m1 = ev->seg_in[a], m2 = ev->seg_out[a], k;
      for (k = byIn[m2]; k < byIn[m2 + 1]; ++k) {
        int32_t b = lst[k], m3 = ev->seg_out[b];
        real p1[4] = { ev->md_x[m1], ev->md_y[m1], ev->md_z[m1], ev->md_r[m1] };
        real p2[4] = { ev->md_x[m2], ev->md_y[m2], ev->md_z[m2], ev->md_r[m2] };
        real p3[4] = { ev->md_x[m3], ev->md_y[m3], ev->md_z[m3], ev->md_r[m3] };
        real out[2];
        ev->cand[2]++;
        if (lsto_t3_cut(cfg, layer[ev->md_module[m1]], p1, p2, p3, out, NULL)) {
          GROW_T3(ev);
          ev->t3_a[ev->n_t3] = (int32_t)a; ev->t3_b[ev->n_t3] = b;
          ev->t3_kappa[ev->n_t3] = out[0]; ev->t3_chi2rz[ev->n_t3] = out[1];
          ev->n_t3++;
        }
      }
    }
    free(byIn); free(lst); free(cur);
  }
  if (stages < 4) return ev;

  /* ---- quintuplets: triplet pairs (A, B) with last MD of A == first MD of B ---- */
  {
    int32_t* byFirst = calloc((size_t)ev->n_md + 1, 4);  /* triplets grouped by first MD */
    int32_t* lst = malloc((size_t)(ev->n_t3 > 0 ? ev->n_t3 : 1) * 4);
    int32_t* cur = calloc((size_t)ev->n_md + 1, 4);
    int64_t t;
    for (t = 0; t < ev->n_t3; ++t) byFirst[ev->seg_in[ev->t3_a[t]] + 1]++;
    for (a = 0; a < ev->n_md; ++a) byFirst[a + 1] += byFirst[a];
    for (t = 0; t < ev->n_t3; ++t) { int32_t i = ev->seg_in[ev->t3_a[t]]; lst[byFirst[i] + cur[i]++] = (int32_t)t; }
    for (t = 0; t < ev->n_t3; ++t) {
      int32_t md[5], k, j;
      md[0] = ev->seg_in[ev->t3_a[t]]; md[1] = ev->seg_out[ev->t3_a[t]]; md[2] = ev->seg_out[ev->t3_b[t]];
      for (k = byFirst[md[2]]; k < byFirst[md[2] + 1]; ++k) {
        int32_t B = lst[k];
        real p[20], out[3];
        md[3] = ev->seg_out[ev->t3_a[B]]; md[4] = ev->seg_out[ev->t3_b[B]];
        for (j = 0; j < 5; ++j) {
          p[4 * j + 0] = ev->md_x[md[j]]; p[4 * j + 1] = ev->md_y[md[j]];
          p[4 * j + 2] = ev->md_z[md[j]]; p[4 * j + 3] = ev->md_r[md[j]];
        }
        ev->cand[3]++;
        if (lsto_t5_cut(cfg, layer[ev->md_module[md[0]]], ev->t3_kappa[t], ev->t3_kappa[B], p, out, NULL)) {
          GROW_T5(ev);
          ev->t5_a[ev->n_t5] = (int32_t)t; ev->t5_b[ev->n_t5] = B;
          ev->t5_kfit[ev->n_t5] = out[0]; ev->t5_chi2xy[ev->n_t5] = out[1]; ev->t5_chi2rz[ev->n_t5] = out[2];
          ev->n_t5++;
        }
      }
    }
    free(byFirst); free(lst); free(cur);
  }
  return ev;
}

/* [P] event level: every (outer object, seed) pair is a candidate -- the search space is the full product, there is no
 * map for seeds -- for the triplets whose innermost layer is 0 or 1 (kind 0) and for all quintuplets (kind 1).  Links come
 * out ordered by (outer object, seed).  Adds to `ev` (built up to stage 3 resp. 4 by lsto_run); returns the number of links. */
int64_t lsto_pixel_link(const lsto_config* cfg, lsto_event* ev, const int8_t* layer, int kind, int32_t n_seeds,
                        const float* kappa, const float* cphi, const float* sphi, const float* z0, const float* t) {
  const int n = kind ? 5 : 3;
  const int64_t n_obj = kind ? ev->n_t5 : ev->n_t3;
  int64_t o;
  int32_t s;
  ev->n_pix[kind] = 0;
  ev->cand_pix[kind] = 0;
  for (o = 0; o < n_obj; ++o) {
    int32_t md[5];
    real p[20], kobj;
    int j, layer1;
    if (kind) {
      const int32_t A = ev->t5_a[o], B = ev->t5_b[o];
      md[0] = ev->seg_in[ev->t3_a[A]]; md[1] = ev->seg_out[ev->t3_a[A]]; md[2] = ev->seg_out[ev->t3_b[A]];
      md[3] = ev->seg_out[ev->t3_a[B]]; md[4] = ev->seg_out[ev->t3_b[B]];
      kobj = ev->t5_kfit[o];
    } else {
      md[0] = ev->seg_in[ev->t3_a[o]]; md[1] = ev->seg_out[ev->t3_a[o]]; md[2] = ev->seg_out[ev->t3_b[o]];
      kobj = ev->t3_kappa[o];
    }
    layer1 = layer[ev->md_module[md[0]]];
    if (layer1 > 1) continue;
    for (j = 0; j < n; ++j) {
      p[4 * j + 0] = ev->md_x[md[j]]; p[4 * j + 1] = ev->md_y[md[j]];
      p[4 * j + 2] = ev->md_z[md[j]]; p[4 * j + 3] = ev->md_r[md[j]];
    }
    for (s = 0; s < n_seeds; ++s) {
      real seed[5], out[3];
      seed[0] = kappa[s]; seed[1] = cphi[s]; seed[2] = sphi[s]; seed[3] = z0[s]; seed[4] = t[s];
      ev->cand_pix[kind]++;
      if (lsto_pix_cut(cfg, kind, layer1, n, seed, kobj, p, out, NULL)) {
        if (ev->n_pix[kind] == ev->cap_pix[kind]) {
          const int64_t c = ev->cap_pix[kind] ? 2 * ev->cap_pix[kind] : 1024;
          ev->pix_seed[kind] = grow(ev->pix_seed[kind], c, 4); ev->pix_obj[kind] = grow(ev->pix_obj[kind], c, 4);
          ev->pix_chi2xy[kind] = grow(ev->pix_chi2xy[kind], c, sizeof(real)); ev->pix_chi2rz[kind] = grow(ev->pix_chi2rz[kind], c, sizeof(real));
          ev->pix_dk[kind] = grow(ev->pix_dk[kind], c, sizeof(real));
          ev->cap_pix[kind] = c;
        }
        ev->pix_seed[kind][ev->n_pix[kind]] = s; ev->pix_obj[kind][ev->n_pix[kind]] = (int32_t)o;
        ev->pix_chi2xy[kind][ev->n_pix[kind]] = out[0]; ev->pix_chi2rz[kind][ev->n_pix[kind]] = out[1];
        ev->pix_dk[kind][ev->n_pix[kind]] = out[2];
        ev->n_pix[kind]++;
      }
    }
  }
  return ev->n_pix[kind];
}
int64_t lsto_pix_count(const lsto_event* ev, int kind) { return ev->n_pix[kind]; }
int64_t lsto_pix_candidates(const lsto_event* ev, int kind) { return ev->cand_pix[kind]; }
const int32_t* lsto_pix_i32(const lsto_event* ev, int kind, int field) { return field ? ev->pix_obj[kind] : ev->pix_seed[kind]; }
const real* lsto_pix_real(const lsto_event* ev, int kind, int field) {
  return field == 0 ? ev->pix_chi2xy[kind] : field == 1 ? ev->pix_chi2rz[kind] : ev->pix_dk[kind];
}

/* ------------------------------------------------------------------------------------ */
/* [D] duplicate cleaning of quintuplets  (DESIGN.md section 1 [D])      */
/* ------------------------------------------------------------------------------------ */
/* The paper cleans duplicates when the track-candidate collection is assembled (PAPER.md:67
 * "cross-clean", :105 "efficient cross-cleaning ... duplicate rates are quite low") and gives no
 * rule for quintuplets among themselves; the rule here is DESIGN.md reading 24:
 *   score(q)  = chi2xy(q) + chi2rz(q)                        (one addition in `real`)
 *   shared(a, b) = number of original hit indices the two quintuplets have in common
 *   b beats a  iff  score(b) < score(a), or the scores are equal and b's hit tuple (10 indices,
 *                   in layer order: MD1 lower, MD1 upper, ...) is lexicographically smaller
 *   a is REMOVED iff some b != a has shared(a, b) >= min_shared and b beats a
 * (removed quintuplets still remove others: the rule is one pass over all pairs, independent of
 * any processing order).  This is the plain definition: every pair is looked at; the common hits
 * of a pair are counted by merging the two sorted copies of the tuples (the 10 hits of a
 * quintuplet are distinct, pin P9).
 * hits: [n][10] original hit indices; keep: [n] out, 1 = kept.  Returns the number kept. */
static int cmp_i32(const void* a, const void* b) {
  const int32_t x = *(const int32_t*)a, y = *(const int32_t*)b;
  return (x > y) - (x < y);
}
int64_t lsto_t5_clean(int64_t n, const int32_t* hits, const real* chi2xy, const real* chi2rz, int min_shared,
                      uint8_t* keep) {
  int64_t a, b, kept = 0;
  int k;
  int32_t* sorted = malloc((size_t)(n > 0 ? n : 1) * 10 * sizeof(int32_t));
  real* score = malloc((size_t)(n > 0 ? n : 1) * sizeof(real));
  for (a = 0; a < n; ++a) {
    for (k = 0; k < 10; ++k) sorted[10 * a + k] = hits[10 * a + k];
    qsort(sorted + 10 * a, 10, sizeof(int32_t), cmp_i32);
    score[a] = chi2xy[a] + chi2rz[a];
    keep[a] = 1;
  }
  for (a = 0; a < n; ++a) {
    for (b = 0; b < n; ++b) {
      int i = 0, j = 0, shared = 0, beats;
      const int32_t *sa = sorted + 10 * a, *sb = sorted + 10 * b;
      if (b == a) continue;
      while (i < 10 && j < 10) {
        if (sa[i] < sb[j]) ++i;
        else if (sa[i] > sb[j]) ++j;
        else { ++shared; ++i; ++j; }
      }
      if (shared < min_shared) continue;
      if (score[b] < score[a]) beats = 1;
      else if (score[b] > score[a]) beats = 0;
      else {
        beats = 0;
        for (k = 0; k < 10; ++k) {
          if (hits[10 * b + k] != hits[10 * a + k]) { beats = hits[10 * b + k] < hits[10 * a + k]; break; }
        }
      }
      if (beats) { keep[a] = 0; break; }
    }
    kept += keep[a];
  }
  free(sorted);
  free(score);
  return kept;
}

/* ------------------------------------------------------------------------------------ */
/* [B] module-map builder  (DESIGN.md section 1 [B])        */
/* ------------------------------------------------------------------------------------ */
/* "derived from first principles by computing the possible track trajectories as helices that can start
 * from the edges of a given module that are compatible with the pT threshold, and then listing all the
 * modules in the adjacent layer that intersect these helices".  The paper gives no
 * formula; the reading (reading 25) is the closed-form envelope of those
 * helices, always in double precision, for a source module A and a module B of the next layer:
 *   radii reached on A / B:  r_lo = rho_A - gap_A/2, r_hi = hypot(rho_A + gap_A/2, hw_A),
 *                            r'_lo = rho_B - gap_B/2, r'_hi = hypot(rho_B + gap_B/2, hw_B)
 *   tightest helix:          R_m = pt_min / (k B), a(r) = asin(min(1, r / (2 R_m)))
 *   azimuth:  |wrap(phi_B - phi_A)| <= atan(hw_A / r_lo) + atan(hw_B / r'_lo) + (a(r'_hi) - a(r_lo)) + pad_phi
 *   z:        the interval spanned by z0 + (z_A - z0) * ratio over z0 in {-z0_max, +z0_max},
 *             z_A in {zlo_A - pad_z, zhi_A + pad_z}, ratio in {r'_lo / r_hi (straight, shortest lever),
 *             a(r'_hi) / a(r_lo) (tightest helix, arc-length ratio)} must meet [zlo_B, zhi_B].
 * rows come out ascending.  counts[n] / targets: the caller passes targets == NULL to count only.
 * Returns the number of connections. */
int64_t lsto_build_map(int32_t n, const int8_t* layer, const double* phi, const double* rho, const double* gap,
                       const double* hw, const double* zlo, const double* zhi, double pt_min, double b_tesla,
                       double z0_max, double pad_phi, double pad_z, int32_t* row_offsets, int32_t* targets) {
  const double kGeV = 2.99792458e-3, kPi = 3.14159265358979323846;
  const double Rm = pt_min / (kGeV * b_tesla);
  int64_t total = 0;
  int32_t A, B;
  for (A = 0; A < n; ++A) {
    row_offsets[A] = (int32_t)total;
    for (B = 0; B < n; ++B) {
      double r_lo, r_hi, rp_lo, rp_hi, a_out, a_in, tol, d, ratio[2], z_lo = 0, z_hi = 0;
      int iz0, iza, ir, first = 1;
      if (layer[B] != layer[A] + 1) continue;
      r_lo = rho[A] - gap[A] / 2;
      r_hi = hypot(rho[A] + gap[A] / 2, hw[A]);
      rp_lo = rho[B] - gap[B] / 2;
      rp_hi = hypot(rho[B] + gap[B] / 2, hw[B]);
      a_out = asin(fmin(1.0, rp_hi / (2 * Rm)));
      a_in = asin(fmin(1.0, r_lo / (2 * Rm)));
      tol = atan(hw[A] / r_lo) + atan(hw[B] / rp_lo) + (a_out - a_in) + pad_phi;
      d = fmod(phi[B] - phi[A], 2 * kPi);            /* into (-pi, pi] */
      if (d > kPi) d -= 2 * kPi;
      if (d <= -kPi) d += 2 * kPi;
      if (!(fabs(d) <= tol)) continue;
      ratio[0] = rp_lo / r_hi;
      ratio[1] = a_out / a_in;
      for (iz0 = 0; iz0 < 2; ++iz0)
        for (iza = 0; iza < 2; ++iza)
          for (ir = 0; ir < 2; ++ir) {
            const double z0 = iz0 ? z0_max : -z0_max;
            const double za = iza ? zhi[A] + pad_z : zlo[A] - pad_z;
            const double zp = z0 + (za - z0) * ratio[ir];
            if (first || zp < z_lo) z_lo = zp;
            if (first || zp > z_hi) z_hi = zp;
            first = 0;
          }
      if (!(z_hi >= zlo[B] && z_lo <= zhi[B])) continue;
      if (targets) targets[total] = B;
      ++total;
    }
  }
  row_offsets[n] = (int32_t)total;
  return total;
}

/* ------------------------------------------------------------------------------------ */
/* [H] reduced-precision object store  (DESIGN.md section 1 [H])        */
/* ------------------------------------------------------------------------------------ */
/* The paper names half precision as future work ("exploring data types such as half precision
 * floats"); the reading (reading 27) stores the per-object OUTPUT floats that no later selection reads as
 * IEEE 754 binary16, each the value nearest to the fp32 result, ties to even; overflow goes to infinity, values
 * below the smallest subnormal to (signed) zero, NaN stays NaN.  This is that rounding, on the bit patterns, so that it
 * does not depend on the compiler's or the CPU's half-precision support.  Pin P21: equals numpy's float32 -> float16
 * conversion on every binary16 value, on every tie and on random inputs (tests/test_oracle_half.py). */
uint16_t lsto_half_bits(float f) {
  uint32_t x, sign, e, m, q, rem, half;
  int shift;
  memcpy(&x, &f, 4);
  sign = (x >> 16) & 0x8000u;
  x &= 0x7fffffffu;
  if (x > 0x7f800000u) return (uint16_t)(sign | 0x7e00u | ((x >> 13) & 0x1ffu));   /* NaN (quiet, payload kept) */
  if (x >= 0x477ff000u) return (uint16_t)(sign | 0x7c00u);   /* >= 65520 = max half + half an ulp: infinity */
  e = x >> 23;
  if (e < 113u) {                                             /* below 2^-14: subnormal half, unit 2^-24 */
    if (e < 102u) return (uint16_t)sign;                      /* below 2^-25: zero */
    m = (x & 0x7fffffu) | 0x800000u;
    shift = (int)(126u - e);                                  /* 14 .. 24 */
    q = m >> shift;
    rem = m & ((1u << shift) - 1u);
    half = 1u << (shift - 1);
  } else {
    m = x & 0x7fffffu;
    q = ((e - 112u) << 10) | (m >> 13);
    rem = m & 0x1fffu;
    half = 0x1000u;
  }
  if (rem > half || (rem == half && (q & 1u))) ++q;           /* nearest, ties to even; a carry moves to the next binade */
  return (uint16_t)(sign | q);
}
void lsto_half_bits_array(int64_t n, const float* in, uint16_t* out) {
  int64_t i;
  for (i = 0; i < n; ++i) out[i] = lsto_half_bits(in[i]);
}

/* ---- accessors for the ctypes wrapper ---- */
int64_t lsto_count(const lsto_event* ev, int kind) {
  switch (kind) { case 0: return ev->n_md; case 1: return ev->n_seg; case 2: return ev->n_t3; case 3: return ev->n_t5; }
  return -1;
}
int64_t lsto_candidates(const lsto_event* ev, int stage) { return (stage >= 0 && stage < 4) ? ev->cand[stage] : -1; }

const int32_t* lsto_i32(const lsto_event* ev, int field) {
  switch (field) {
    case 0: return ev->md_lower; case 1: return ev->md_upper; case 2: return ev->md_module;
    case 3: return ev->seg_in;   case 4: return ev->seg_out;
    case 5: return ev->t3_a;     case 6: return ev->t3_b;
    case 7: return ev->t5_a;     case 8: return ev->t5_b;
  }
  return NULL;
}
const real* lsto_real(const lsto_event* ev, int field) {
  switch (field) {
    case 0: return ev->md_x; case 1: return ev->md_y; case 2: return ev->md_z; case 3: return ev->md_r;
    case 4: return ev->md_ur; case 5: return ev->md_sinA; case 6: return ev->md_dphi; case 7: return ev->md_dphichange;
    case 8: return ev->seg_sinS; case 9: return ev->seg_z0; case 10: return ev->seg_dphi; case 11: return ev->seg_dphichange;
    case 12: return ev->t3_kappa; case 13: return ev->t3_chi2rz;
    case 14: return ev->t5_kfit; case 15: return ev->t5_chi2xy; case 16: return ev->t5_chi2rz;
  }
  return NULL;
}
