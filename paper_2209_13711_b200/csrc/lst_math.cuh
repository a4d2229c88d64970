// lst_math.cuh -- per-candidate selection arithmetic of the CUDA path (DESIGN.md Readings C0-C6).
//
// Two flavours per object level:
//   *_pre_f : fp32 conservative pre-filter.  It may only REJECT a candidate whose cut variable
//             exceeds the threshold by more than PRE_SLACK (1e-3 relative), far outside the fp32
//             evaluation error of the difference-first formulas; NaN never rejects.
//   *_d     : fp64 decision on the fp32 inputs promoted before the first subtraction, and the
//             derived quantities that are stored.  Every accepted object is decided here.
// Functions are __host__ __device__ so that the host test hooks (lst_host_* in lst_api.cu) can run
// the very same code on the CPU.  Nothing here is shared with oracle/.
#pragma once
#include <math.h>
#include <stdint.h>

#ifdef __CUDACC__
#define LST_HD __host__ __device__ __forceinline__
#else
#define LST_HD inline
#endif

namespace lst {

constexpr double kGuard = 1e-9;       // denominators must exceed this (C0)
constexpr float kPreSlack = 1.001f;   // fp32 pre-filter loosening

// Division inside the fp32 pre-filters: the 2-ulp approximate divide on the device (the pre-filters
// are loosened by 1e-3 relative, 4 orders of magnitude more), the plain one on the host.
#ifdef __CUDA_ARCH__
#define LST_FDIV(a, b) __fdividef((a), (b))
#else
#define LST_FDIV(a, b) ((a) / (b))
#endif

// Selection parameters in the form the kernels use (built once by lst_create from lst_config).
struct Params {
  double kmax;          // kB / (2 pt_min)
  double kB, ns, z0max, d0max, chi2max, dr2max, ec_md_sys, modez_slack;
  double seed_sig_phi, seed_sig_pt, seed_sig_z;
  double sig_t[4], sig_z[4], sig_r[4];
  float f_kmax, f_ns, f_z0max, f_ec_md_sys, f_modez_slack;
  float f_sig_t[4], f_sig_z[4], f_sig_r[4];
  int dup_t5, dup_pt5, dup_pt3, s0_enabled;
  uint32_t start_mask;
  // eta binning of the pixel seeds used by the cleaning (k_dedup.cu)
  double eta_bin_inv, dr_eta_pre;
  int eta_nbins;
  uint32_t trunc[6][16];   // occupancy truncation (lst_config.trunc_cap): per lst_level and logical layer, 0 = none
};

LST_HD bool is_endcap(int cat) { return cat >= 2; }
LST_HD double clamp1(double v) { return v > 1.0 ? 1.0 : (v < -1.0 ? -1.0 : v); }
LST_HD double dmin(double a, double b) { return a < b ? a : b; }
LST_HD double wrap_pi(double a) { return remainder(a, 6.283185307179586476925286766559); }
// sqrt(a^2 + b^2): coordinates are centimetres (|a|, |b| < 1e4), so no overflow / underflow handling.
LST_HD double hyp(double a, double b) { return sqrt(a * a + b * b); }
// atan2 for the small angles between neighbouring anchors (every LS has |sin dphi| <~ 0.2 and a
// positive dot product): for x > 0, |y| <= x / 4 the odd series in t = y / x, 11 terms, truncation
// error < 3e-15 relative; anything else goes to libm.  The north_star contract needs cut variables
// to 1e-5 of their thresholds, which this exceeds by ten orders of magnitude.
LST_HD double atan2_small(double y, double x) {
  if (x > 0.0 && fabs(y) <= 0.25 * x) {
    const double t = y / x, u = t * t;
    double p = 1.0 / 21.0;
    p = -1.0 / 19.0 + u * p;
    p = 1.0 / 17.0 + u * p;
    p = -1.0 / 15.0 + u * p;
    p = 1.0 / 13.0 + u * p;
    p = -1.0 / 11.0 + u * p;
    p = 1.0 / 9.0 + u * p;
    p = -1.0 / 7.0 + u * p;
    p = 1.0 / 5.0 + u * p;
    p = -1.0 / 3.0 + u * p;
    p = 1.0 + u * p;
    return t * p;
  }
  return atan2(y, x);
}

struct Pt {  // a point promoted to double, with its transverse radius and module category
  double x, y, z, rt;
  int cat;
};
LST_HD Pt make_pt(float x, float y, float z, int cat) {
  Pt p;
  p.x = (double)x; p.y = (double)y; p.z = (double)z;
  p.rt = sqrt(p.x * p.x + p.y * p.y);
  p.cat = cat;
  return p;
}
// C0 helpers (difference first)
LST_HD double sd_of(const Pt &A, const Pt &B) {          // sin(dphi)
  return (A.x * (B.y - A.y) - A.y * (B.x - A.x)) / (A.rt * B.rt);
}
LST_HD double dphi_of(const Pt &A, const Pt &B) {
  return atan2_small(A.x * (B.y - A.y) - A.y * (B.x - A.x), A.x * B.x + A.y * B.y);
}
LST_HD double chord_of(const Pt &A, const Pt &B) { return hyp(B.x - A.x, B.y - A.y); }
LST_HD double dr_of(const Pt &A, const Pt &B) {          // rt_B - rt_A without cancellation
  double dx = B.x - A.x, dy = B.y - A.y;
  return (2.0 * (A.x * dx + A.y * dy) + (dx * dx + dy * dy)) / (A.rt + B.rt);
}
LST_HD double kappa3_of(const Pt &A, const Pt &B, const Pt &C) {  // Menger curvature / 2
  double abx = B.x - A.x, aby = B.y - A.y, bcx = C.x - B.x, bcy = C.y - B.y;
  double acx = C.x - A.x, acy = C.y - A.y;
  return (abx * bcy - aby * bcx) / (hyp(abx, aby) * hyp(bcx, bcy) * hyp(acx, acy));
}
LST_HD double arc_of(double r, double k) {               // arc length at radius r, half curvature k
  if (fabs(k * r) <= 1e-4) return r;
  return asin(clamp1(k * r)) / k;
}
// "v <= thr" with NaN failing
LST_HD bool le(double v, double thr) { return v <= thr; }

// fp32 atan2 for the pre-filters: for x > 0, |y| <= x / 4 the odd series in t = y / x to t^11
// (truncation < 2e-9 relative, below the fp32 rounding of the result); atan2f otherwise.
LST_HD float atan2_small_f(float y, float x) {
  if (x > 0.0f && fabsf(y) <= 0.25f * x) {
    const float t = LST_FDIV(y, x), u = t * t;
    return t * (1.0f + u * (-0.33333333f + u * (0.2f + u * (-0.14285714f + u * (0.11111111f - 0.09090909f * u)))));
  }
  return atan2f(y, x);
}

// ------------------------------------------------------------------ C1 mini-doublet
struct MdOut { double kappa, sigk, dphi; };

LST_HD bool md_eval_d(const Params &g, const Pt &l, const Pt &u, int cat, MdOut *o) {
  if (!(l.rt > kGuard) || !(u.rt > kGuard)) return false;
  const double dz = u.z - l.z;
  const double sdv = sd_of(l, u), cxy = chord_of(l, u), drv = dr_of(l, u);
  const double st = g.sig_t[cat];
  const double inv = 1.0 / l.rt + 1.0 / u.rt;
  const double tolphi = g.ns * st * inv;
  bool ok = true;
  double cpred;
  if (!is_endcap(cat)) {
    ok &= (drv > 0.0);                                                                         // B1
    ok &= le(fabs(dz - l.z * drv / l.rt), g.z0max * drv / l.rt + 2.0 * g.ns * g.sig_z[cat]);
    ok &= le(fabs(sdv), g.kmax * cxy + tolphi);                                                // B2
    cpred = cxy;
  } else {
    const double azl = fabs(l.z);
    if (!(azl > kGuard) || !(azl - g.z0max > kGuard)) return false;
    ok &= le(fabs(drv - l.rt * dz / l.z),                                                      // E1
             l.rt * fabs(dz) * g.z0max / (azl * (azl - g.z0max)) + 2.0 * g.ns * g.sig_r[cat]);
    ok &= le(fabs(sdv), fabs(dz) * asin(dmin(1.0, g.kmax * l.rt)) / (azl - g.z0max) + tolphi);  // E2
    cpred = fabs(dz) * l.rt / azl;
  }
  if (!(cpred > kGuard)) return false;
  if (o) {
    o->kappa = sdv / cpred;
    o->sigk = st * inv / cpred;
    o->dphi = asin(clamp1(sdv));
  }
  return ok;
}

// fp32 pre-filter: true = keep for the fp64 decision.  rt* are fp32 sqrt(x^2+y^2).
LST_HD bool md_pre_f(const Params &g, float xl, float yl, float zl, float rl, float xu, float yu, float zu,
                     float ru, int cat) {
  const float dx = xu - xl, dy = yu - yl, dz = zu - zl;
  const float dd = dx * dx + dy * dy;
  const float drv = LST_FDIV(2.0f * (xl * dx + yl * dy) + dd, rl + ru);
  const float cr = xl * dy - yl * dx;
  const float tolrr = g.f_ns * g.f_sig_t[cat] * (rl + ru);       // tolphi * rl * ru
  const float rr = rl * ru;
  if (!is_endcap(cat)) {
    if (drv < -1e-3f) return false;
    const float t = LST_FDIV(drv, rl);
    if (fabsf(dz - zl * t) > (g.f_z0max * t + 2.0f * g.f_ns * g.f_sig_z[cat]) * kPreSlack + 1e-4f) return false;
    if (fabsf(cr) > (g.f_kmax * sqrtf(dd) * rr + tolrr) * kPreSlack) return false;
  } else {
    const float azl = fabsf(zl);
    const float den = azl - g.f_z0max;
    if (den < 1e-3f) return true;  // let the fp64 guard decide
    const float adz = fabsf(dz);
    if (fabsf(drv - LST_FDIV(rl * dz, zl)) > (LST_FDIV(rl * adz * g.f_z0max, azl * den) + 2.0f * g.f_ns * g.f_sig_r[cat]) * kPreSlack + 1e-4f)
      return false;
    const float asl = asinf(fminf(1.0f, g.f_kmax * rl));
    if (fabsf(cr) > (LST_FDIV(adz * asl, den) * rr + tolrr) * kPreSlack) return false;
  }
  return true;
}

// ------------------------------------------------------------------ C3 line segment
struct LsOut { double kappa, sigk, dphi; };

// A, B: anchors of the inner / outer MD; (ki, ski), (ko, sko): their kappa_MD, sigma_kappa_MD.
LST_HD bool ls_eval_d(const Params &g, const Pt &A, double ki, double ski, const Pt &B, double ko, double sko,
                      LsOut *o) {
  const int ci = A.cat, co = B.cat;
  const bool modeZ = is_endcap(co);
  const double ns = g.ns;
  const double dz = B.z - A.z;
  const double drv = dr_of(A, B), sdv = sd_of(A, B), cxy = chord_of(A, B), dph = dphi_of(A, B);
  bool ok = true;
  // L1 pointing
  const double N = A.rt * dz - A.z * drv;
  const double E = A.rt * g.sig_z[co] + B.rt * g.sig_z[ci] + fabs(B.z) * g.sig_r[ci] + fabs(A.z) * g.sig_r[co];
  ok &= le(fabs(N), g.z0max * fabs(drv) + ns * E);
  // L2 pT window
  const double tphi = g.sig_t[ci] / A.rt + g.sig_t[co] / B.rt;
  const double tolphi = ns * tphi;
  ok &= (A.x * B.x + A.y * B.y > 0.0);
  double kls, sigkls, slack;
  if (!modeZ) {
    if (!(cxy > kGuard)) return false;
    ok &= le(fabs(sdv), g.kmax * cxy + tolphi);
    kls = sdv / cxy;
    sigkls = tphi / cxy;
    slack = 0.0;
  } else {
    const double rbar = 0.5 * (A.rt + B.rt), zbar = 0.5 * (fabs(A.z) + fabs(B.z));
    const double adz = fabs(dz);
    if (!(adz > kGuard) || !(rbar > kGuard)) return false;
    const double Sbar = asin(dmin(1.0, g.kmax * (rbar + ns * (g.sig_r[ci] + g.sig_r[co]) / 2.0))) / g.kmax;
    const double den = zbar - g.z0max - ns * g.sig_z[ci] / 2.0;
    if (!(den > kGuard)) return false;
    ok &= le(fabs(dph), g.kmax * (adz + ns * g.sig_z[ci]) * Sbar / den + tolphi);
    const double lever = zbar / (adz * rbar);
    kls = dph * lever;
    sigkls = tphi * lever;
    slack = fabs(kls) * (g.z0max / zbar + g.modez_slack + ns * (g.sig_r[ci] + g.sig_r[co]) / (A.rt + B.rt) +
                         ns * g.sig_z[ci] / adz);
  }
  // L3 stub-segment curvature consistency
  ok &= le(fabs(ki - kls), ns * (ski + sigkls) + slack + (is_endcap(ci) ? g.ec_md_sys * fabs(kls) : 0.0));
  ok &= le(fabs(ko - kls), ns * (sko + sigkls) + slack + (is_endcap(co) ? g.ec_md_sys * fabs(kls) : 0.0));
  if (o) { o->kappa = kls; o->sigk = sigkls; o->dphi = dph; }
  return ok;
}

// Tier 2 of the LS pre-filter (full fp32 L2 and L3).  It runs on candidates that passed tier 1
// (ls_tier1_f: pointing L1 and the positive dot product), which it does not repeat.
LST_HD bool ls_pre_f(const Params &g, float xi, float yi, float zi, float ri, float ki, float ski, int ci,
                     float xo, float yo, float zo, float ro, float ko, float sko, int co) {
  const float ns = g.f_ns;
  const float rr = ri * ro;
  const float cr = xi * yo - yi * xo;       // cross(A, D) = cross(A, B)
  const float sd = LST_FDIV(cr, rr);
  const float tphi = LST_FDIV(g.f_sig_t[ci], ri) + LST_FDIV(g.f_sig_t[co], ro);
  const float eci = is_endcap(ci) ? g.f_ec_md_sys : 0.0f, eco = is_endcap(co) ? g.f_ec_md_sys : 0.0f;
  if (!is_endcap(co)) {
    const float dx = xo - xi, dy = yo - yi;
    const float cxy = sqrtf(dx * dx + dy * dy);
    const float asd = fabsf(sd);
    if (asd > (g.f_kmax * cxy + ns * tphi) * kPreSlack) return false;
    // L3 multiplied through by cxy
    if (fabsf(ki * cxy - sd) > (ns * (ski * cxy + tphi) + eci * asd) * kPreSlack) return false;
    if (fabsf(ko * cxy - sd) > (ns * (sko * cxy + tphi) + eco * asd) * kPreSlack) return false;
  } else {
    const float rbar = 0.5f * (ri + ro), zbar = 0.5f * (fabsf(zi) + fabsf(zo));
    const float adz = fabsf(zo - zi);
    const float den = zbar - g.f_z0max - 0.5f * ns * g.f_sig_z[ci];
    if (den < 1e-3f || adz < 1e-6f) return true;   // guards are decided in fp64
    const float srs = g.f_sig_r[ci] + g.f_sig_r[co];
    // asin(x) <= x + (pi/2 - 1) x^3 on [0, 1]: an upper bound only loosens the L2 window
    const float xs = fminf(1.0f, g.f_kmax * (rbar + 0.5f * ns * srs));
    const float Sbar = LST_FDIV(xs + 0.5708f * xs * xs * xs, g.f_kmax);
    // dphi = atan2(cr, dot): for |cr| <= dot / 2 the odd series to t^11 (error < 1e-5 relative)
    const float dotAB = xi * xo + yi * yo;
    float dph;
    if (dotAB > 0.0f && fabsf(cr) <= 0.5f * dotAB) {
      const float t = LST_FDIV(cr, dotAB), u = t * t;
      dph = t * (1.0f + u * (-0.33333333f + u * (0.2f + u * (-0.14285714f + u * (0.11111111f - 0.09090909f * u)))));
    } else {
      dph = atan2f(cr, dotAB);
    }
    if (fabsf(dph) > (LST_FDIV(g.f_kmax * (adz + ns * g.f_sig_z[ci]) * Sbar, den) + ns * tphi) * kPreSlack) return false;
    const float lever = LST_FDIV(zbar, adz * rbar);
    const float kls = dph * lever, akls = fabsf(kls);
    const float sigkls = tphi * lever;
    const float slack = akls * (LST_FDIV(g.f_z0max, zbar) + g.f_modez_slack + LST_FDIV(ns * srs, ri + ro) + LST_FDIV(ns * g.f_sig_z[ci], adz));
    if (fabsf(ki - kls) > (ns * (ski + sigkls) + slack + eci * akls) * kPreSlack) return false;
    if (fabsf(ko - kls) > (ns * (sko + sigkls) + slack + eco * akls) * kPreSlack) return false;
  }
  return true;
}

// Tier-1 LS pre-filter: cuts L1 (pointing) and L2 (pT window) multiplied through by their positive
// denominators, so no division, square root or inverse trigonometric function is evaluated; the
// mode-Z window uses |sin dphi| <= |dphi| and asin(x) <= x + (pi/2 - 1) x^3 on [0, 1].  It is a
// NECESSARY condition of ls_pre_f (looser), hence of the fp64 decision.  t*: {sig_z, sig_r, sig_t}
// of the inner (i) / outer (o) MD's module category; oec: outer module is an endcap module.
LST_HD bool ls_tier1_f(const Params &g, float xi, float yi, float zi, float ri, float szi, float sri, float sti,
                       float xo, float yo, float zo, float ro, float szo, float sro, float sto, bool oec) {
  // L1: rt_i dz - z_i drv with drv = rt_o - rt_i is the r-z cross product rt_i z_o - z_i rt_o
  // (the fp32 error of the stored radii, ~1e-5 cm, is 1e-5 of the threshold z0max |drv| >= ~100 cm^2)
  const float ns = g.f_ns;
  const float azi = fabsf(zi), azo = fabsf(zo);
  const float E = ri * szo + ro * szi + azo * sri + azi * sro;
  bool keep = !(fabsf(ri * zo - zi * ro) > (g.f_z0max * fabsf(ro - ri) + ns * E) * kPreSlack);              // L1
  const float rr = ri * ro;
  keep &= !(xi * xo + yi * yo < -1e-3f * rr);
  const float acr = fabsf(xi * yo - yi * xo);   // |cross(A, D)| = |cross(A, B)|
  const float T = ns * (sti * ro + sto * ri);   // tolphi * rr
  if (!oec) {
    const float dx = xo - xi, dy = yo - yi;
    const float dd = dx * dx + dy * dy;
    const float e = acr - T * kPreSlack;
    const float kk = g.f_kmax * kPreSlack;
    keep &= !(e > 0.0f && e * e > kk * kk * dd * rr * rr);                                           // L2, mode R
  } else {
    const float x = fminf(1.0f, g.f_kmax * (0.5f * (ri + ro) + 0.5f * ns * (sri + sro)));
    const float ub = x + 0.5708f * x * x * x;
    const float den = 0.5f * (azi + azo) - g.f_z0max - 0.5f * ns * szi;
    if (den >= 1e-3f) keep &= !(acr * den > ((fabsf(zo - zi) + ns * szi) * ub * rr + T * den) * kPreSlack);   // L2, mode Z
  }
  return keep;
}

// Per-(row MD, connected module) window of the LS enumeration.  (ri, zi, ci): the inner anchor;
// (rlo, rhi, zlo, zhi): bounding box of the ANCHORS of the module's MDs in this event (measured from
// the MDs, so nothing is assumed about the geometry description); cB: the module's category.
// Returns false if NO anchor inside the box can pass cut L1 (interval arithmetic on the bilinear
// r-z cross product: its extremes over the box are at the corners).  Otherwise *W bounds |dphi| of
// every pair that can pass L2 (and dot > 0); *W > pi means "no bound" (whole module):
//   mode R: a passing pair lies on a circle through the origin of half curvature k <= kmax + tol /
//     chord with chord >= rlo - ri; on it dphi = asin(k ro) - asin(k ri) (both points on the outgoing
//     arc: the mixed outgoing / returning case needs asin(k ro) + asin(k ri) > pi/2 to keep dot > 0,
//     impossible for k rhi <= 0.6), increasing in k and in ro;
//   mode Z: L2 is itself a bound on |dphi|, taken at the box extremes.
// Every bound is loosened by 2e-3 relative and 2e-4 rad (fp32 evaluation error ~1e-6); a NaN never
// rejects.  It is a NECESSARY condition of ls_tier1_f, hence of the fp64 decision.
LST_HD bool ls_row_window(const Params &g, float ri, float zi, int ci, float rlo, float rhi, float zlo, float zhi,
                          int cB, float *W) {
  const float ns = g.f_ns;
  const float n1 = ri * zlo - zi * rlo, n2 = ri * zlo - zi * rhi, n3 = ri * zhi - zi * rlo, n4 = ri * zhi - zi * rhi;
  const float nmin = fminf(fminf(n1, n2), fminf(n3, n4)), nmax = fmaxf(fmaxf(n1, n2), fmaxf(n3, n4));
  const float azo = fmaxf(fabsf(zlo), fabsf(zhi));
  const float E = ri * g.f_sig_z[cB] + rhi * g.f_sig_z[ci] + azo * g.f_sig_r[ci] + fabsf(zi) * g.f_sig_r[cB];
  const float dr = fmaxf(fabsf(rhi - ri), fabsf(rlo - ri));
  const float rhs = (g.f_z0max * dr + ns * E) * 1.002f + 0.05f;
  if (nmin > rhs || nmax < -rhs) return false;                                                  // L1
  const float tol = ns * (LST_FDIV(g.f_sig_t[ci], ri) + LST_FDIV(g.f_sig_t[cB], rlo));
  float w = 4.0f;
  if (cB < 2) {
    const float cmin = rlo - ri;
    if (cmin > 1.0f) {
      const float k = (g.f_kmax + LST_FDIV(tol, cmin)) * 1.002f;
      // asin(b) - asin(a) = integral of 1 / sqrt(1 - x^2) over [a, b] <= (b - a) / sqrt(1 - b^2)
      const float bq = k * rhi;
      if (bq <= 0.6f) w = LST_FDIV(bq - k * ri, sqrtf(1.0f - bq * bq)) * 1.002f + 2e-4f;             // L2, mode R
    }
  } else {
    const float azo0 = (zlo <= 0.0f && zhi >= 0.0f) ? 0.0f : fminf(fabsf(zlo), fabsf(zhi));
    const float dzmax = fmaxf(fabsf(zhi - zi), fabsf(zlo - zi));
    const float den = 0.5f * (fabsf(zi) + azo0) - g.f_z0max - 0.5f * ns * g.f_sig_z[ci];
    if (den > 1.0f) {
      const float x = fminf(1.0f, g.f_kmax * (0.5f * (ri + rhi) + 0.5f * ns * (g.f_sig_r[ci] + g.f_sig_r[cB])));
      w = (LST_FDIV((dzmax + ns * g.f_sig_z[ci]) * (x + 0.5708f * x * x * x), den) + tol) * 1.002f + 2e-4f;   // L2, mode Z: asin(x) <= x + (pi/2 - 1) x^3
    }
  }
  *W = w;
  return true;
}

// Mode-R line segments in one fp32 pass (the tier-1 conditions plus L3): for an outer MD in a barrel
// module cut L3, |kappa_MD(m) - kappa_LS| <= N_s (sigma_MD(m) + sigma_LS) + 0.3 |kappa_LS| [m endcap],
// multiplied through by chord * rt_i * rt_o, needs one square root and no division:
//   |k_m c rr - cr| <= N_s (s_m c rr + tphi rr) + ec_m |cr|,   cr = cross(A, B), c = chord, rr = rt_i rt_o.
// Same contract as ls_pre_f (may only reject beyond kPreSlack; NaN never rejects): a mode-R candidate
// that passes ls_tier1_f and this needs no further fp32 test.
LST_HD bool ls_l3_modeR_f(const Params &g, float xi, float yi, float ri, float ki, float ski, float sti, bool iec,
                          float xo, float yo, float ro, float ko, float sko, float sto) {
  const float rr = ri * ro;
  const float cr = xi * yo - yi * xo;
  const float dx = xo - xi, dy = yo - yi;
  const float crr = sqrtf(dx * dx + dy * dy) * rr;
  const float T = g.f_ns * (sti * ro + sto * ri);            // N_s tphi rr
  const float eci = iec ? g.f_ec_md_sys * fabsf(cr) : 0.0f;
  bool keep = !(fabsf(ki * crr - cr) > (g.f_ns * ski * crr + T + eci) * kPreSlack);
  keep &= !(fabsf(ko * crr - cr) > (g.f_ns * sko * crr + T) * kPreSlack);
  return keep;
}

// ------------------------------------------------------------------ C4 triplet
struct T3Out { double kappa3, sigk3, beta; };

LST_HD double sig_perp(const Params &g, const Pt &h) {
  return g.sig_t[h.cat] + g.sig_r[h.cat] * dmin(1.0, g.kmax * h.rt);
}

LST_HD bool t3_eval_d(const Params &g, const Pt &P1, const Pt &P2, const Pt &P3, T3Out *o) {
  const double ns = g.ns;
  const bool modeZ = is_endcap(P1.cat) || is_endcap(P2.cat) || is_endcap(P3.cat);
  const double d12x = P2.x - P1.x, d12y = P2.y - P1.y, d23x = P3.x - P2.x, d23y = P3.y - P2.y;
  const double a = hyp(d12x, d12y), b = hyp(d23x, d23y), c13 = chord_of(P1, P3);
  if (!(a > kGuard) || !(b > kGuard) || !(c13 > kGuard)) return false;
  bool ok = true;
  // T3-1 relative angle
  const double crs = d12x * d23y - d12y * d23x;
  const double k3 = crs / (a * b * c13);
  const double sk3 = (sig_perp(g, P2) + (b * sig_perp(g, P1) + a * sig_perp(g, P3)) / c13) / (a * b);
  ok &= le(fabs(k3), g.kmax + ns * sk3);
  // T3-2 phi-lever linearity
  const double d12 = dphi_of(P1, P2), d23 = dphi_of(P2, P3), d13 = d12 + d23;
  const double k13 = sin(d13) / c13;
  double L1, L2, L3, s1 = 0.0, s2 = 0.0, s3 = 0.0;
  if (modeZ) {
    L1 = P1.z; L2 = P2.z; L3 = P3.z;
    s1 = g.sig_z[P1.cat]; s2 = g.sig_z[P2.cat]; s3 = g.sig_z[P3.cat];
  } else {
    L1 = arc_of(P1.rt, k13); L2 = arc_of(P2.rt, k13); L3 = arc_of(P3.rt, k13);
  }
  const double i1 = 1.0 / P1.rt, i2 = 1.0 / P2.rt, i3 = 1.0 / P3.rt;
  const double Nphi = d12 * (L3 - L2) - d23 * (L2 - L1);
  const double Nrho = (i2 - i1) * (L3 - L2) - (i3 - i2) * (L2 - L1);
  const double Ephi = g.sig_t[P1.cat] * i1 * fabs(L3 - L2) + g.sig_t[P2.cat] * i2 * fabs(L3 - L1) +
                      g.sig_t[P3.cat] * i3 * fabs(L2 - L1) + s1 * fabs(d23) + s2 * fabs(d13) + s3 * fabs(d12);
  ok &= le(fabs(Nphi), g.d0max * fabs(Nrho) + ns * Ephi);
  // T3-3 r-z collinearity
  const double q1 = k3 * P1.rt, q2 = k3 * P2.rt, q3 = k3 * P3.rt;
  const double a1 = P1.rt * (1.0 + q1 * q1 / 6.0), a2 = P2.rt * (1.0 + q2 * q2 / 6.0), a3 = P3.rt * (1.0 + q3 * q3 / 6.0);
  const double Nz = (a2 - a1) * (P3.z - P1.z) - (a3 - a1) * (P2.z - P1.z);
  const double Ez = g.sig_z[P3.cat] * fabs(a2 - a1) + g.sig_z[P2.cat] * fabs(a3 - a1) + g.sig_z[P1.cat] * fabs(a3 - a2) +
                    g.sig_r[P2.cat] * fabs(P3.z - P1.z) + g.sig_r[P3.cat] * fabs(P2.z - P1.z) +
                    g.sig_r[P1.cat] * fabs(P3.z - P2.z);
  ok &= le(fabs(Nz), ns * Ez);
  if (o) {
    o->kappa3 = k3; o->sigk3 = sk3;
    o->beta = atan2_small(crs, d12x * d23x + d12y * d23y);
  }
  return ok;
}

// fp32 pre-filter of a triplet: T3-1 (multiplied through by a b c13, no division) and T3-3, both
// without trigonometry; T3-2 (second differences of angles) is left to the fp64 decision.  Loosened
// by kPreSlack and, for T3-3, an absolute 0.02 cm^2 (fp32 error of N is < 2e-3; N_sigma E >= ~8).
LST_HD bool t3_pre_f(const Params &g, float x1, float y1, float z1, float r1, int c1, float x2, float y2, float z2,
                     float r2, int c2, float x3, float y3, float z3, float r3, int c3) {
  const float d12x = x2 - x1, d12y = y2 - y1, d23x = x3 - x2, d23y = y3 - y2, d13x = x3 - x1, d13y = y3 - y1;
  const float a2 = d12x * d12x + d12y * d12y, b2 = d23x * d23x + d23y * d23y, c2q = d13x * d13x + d13y * d13y;
  if (!(a2 > 1e-10f) || !(b2 > 1e-10f) || !(c2q > 1e-10f)) return true;   // guards are decided in fp64
  const float a = sqrtf(a2), b = sqrtf(b2), c13 = sqrtf(c2q);
  const float crs = d12x * d23y - d12y * d23x;
  const float sp1 = g.f_sig_t[c1] + g.f_sig_r[c1] * fminf(1.0f, g.f_kmax * r1);
  const float sp2 = g.f_sig_t[c2] + g.f_sig_r[c2] * fminf(1.0f, g.f_kmax * r2);
  const float sp3 = g.f_sig_t[c3] + g.f_sig_r[c3] * fminf(1.0f, g.f_kmax * r3);
  const float abc = a * b * c13;
  if (fabsf(crs) > (g.f_kmax * abc + g.f_ns * (sp2 * c13 + b * sp1 + a * sp3)) * kPreSlack) return false;   // T3-1
  const float k3 = LST_FDIV(crs, abc);
  const float q1 = k3 * r1, q2 = k3 * r2, q3 = k3 * r3;
  const float s21 = (r2 - r1) + (r2 * q2 * q2 - r1 * q1 * q1) * (1.0f / 6.0f);
  const float s31 = (r3 - r1) + (r3 * q3 * q3 - r1 * q1 * q1) * (1.0f / 6.0f);
  const float s32 = s31 - s21;
  const float z31 = z3 - z1, z21 = z2 - z1, z32 = z3 - z2;
  const float N = s21 * z31 - s31 * z21;
  const float E = g.f_sig_z[c3] * fabsf(s21) + g.f_sig_z[c2] * fabsf(s31) + g.f_sig_z[c1] * fabsf(s32) +
                  g.f_sig_r[c2] * fabsf(z31) + g.f_sig_r[c3] * fabsf(z21) + g.f_sig_r[c1] * fabsf(z32);
  if (fabsf(N) > g.f_ns * E * kPreSlack + 0.02f) return false;                                              // T3-3
  // T3-2 in fp32: its error (~5e-6, from atan2f / asinf and the products) is three orders of magnitude
  // below the smallest threshold (~5e-3); loosened by 1 % and 2e-4 absolute.
  const float d12 = atan2_small_f(x1 * d12y - y1 * d12x, x1 * x2 + y1 * y2);
  const float d23 = atan2_small_f(x2 * d23y - y2 * d23x, x2 * x3 + y2 * y3);
  const float d13 = d12 + d23;
  float L1, L2, L3, sl1 = 0.0f, sl2 = 0.0f, sl3 = 0.0f;
  if (c1 >= 2 || c2 >= 2 || c3 >= 2) {
    L1 = z1; L2 = z2; L3 = z3;
    sl1 = g.f_sig_z[c1]; sl2 = g.f_sig_z[c2]; sl3 = g.f_sig_z[c3];
  } else {
    const float k13 = LST_FDIV(sinf(d13), c13);
    const float u1 = k13 * r1, u2 = k13 * r2, u3 = k13 * r3;
    L1 = fabsf(u1) <= 1e-4f ? r1 : LST_FDIV(asinf(fminf(1.0f, fmaxf(-1.0f, u1))), k13);
    L2 = fabsf(u2) <= 1e-4f ? r2 : LST_FDIV(asinf(fminf(1.0f, fmaxf(-1.0f, u2))), k13);
    L3 = fabsf(u3) <= 1e-4f ? r3 : LST_FDIV(asinf(fminf(1.0f, fmaxf(-1.0f, u3))), k13);
  }
  const float i1 = LST_FDIV(1.0f, r1), i2 = LST_FDIV(1.0f, r2), i3 = LST_FDIV(1.0f, r3);
  const float L32 = L3 - L2, L21 = L2 - L1, L31 = L3 - L1;
  const float Nphi = d12 * L32 - d23 * L21;
  const float Nrho = (i2 - i1) * L32 - (i3 - i2) * L21;
  const float Ephi = g.f_sig_t[c1] * i1 * fabsf(L32) + g.f_sig_t[c2] * i2 * fabsf(L31) + g.f_sig_t[c3] * i3 * fabsf(L21) +
                     sl1 * fabsf(d23) + sl2 * fabsf(d13) + sl3 * fabsf(d12);
  if (fabsf(Nphi) > ((float)g.d0max * fabsf(Nrho) + g.f_ns * Ephi) * 1.01f + 2e-4f) return false;           // T3-2
  return true;
}

// ------------------------------------------------------------------ C5 quintuplet
struct T5Out { double R, chi2, pt, eta, phi; };

// Weighted Kasa circle fit of 5 points; kc = |kappa3(P1,P3,P5)|.
LST_HD bool kasa_fit_d(const Params &g, const Pt *P, double kc, double *R, double *chi2) {
  double w[5], sw = 0.0, mx = 0.0, my = 0.0;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const double st = g.sig_t[P[k].cat], sr = g.sig_r[P[k].cat] * dmin(1.0, kc * P[k].rt);
    w[k] = 1.0 / (st * st + sr * sr);
    sw += w[k]; mx += w[k] * P[k].x; my += w[k] * P[k].y;
  }
  mx /= sw; my /= sw;
  double u[5], v[5], Suu = 0, Suv = 0, Svv = 0, Suz = 0, Svz = 0, Sz = 0;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    u[k] = P[k].x - mx; v[k] = P[k].y - my;
    const double zeta = u[k] * u[k] + v[k] * v[k];
    Suu += w[k] * u[k] * u[k]; Suv += w[k] * u[k] * v[k]; Svv += w[k] * v[k] * v[k];
    Suz += w[k] * u[k] * zeta; Svz += w[k] * v[k] * zeta; Sz += w[k] * zeta;
  }
  const double det = Suu * Svv - Suv * Suv;
  if (!(det > 0.0)) return false;
  const double Bc = (-Suz * Svv + Svz * Suv) / det;
  const double Cc = (-Svz * Suu + Suz * Suv) / det;
  const double cx = -Bc / 2.0, cy = -Cc / 2.0;
  const double R2 = (Bc * Bc + Cc * Cc) / 4.0 + Sz / sw;
  if (!(R2 > 0.0)) return false;
  const double Rr = sqrt(R2);
  double x2 = 0.0;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const double e = hyp(u[k] - cx, v[k] - cy) - Rr;
    x2 += w[k] * e * e;
  }
  *R = Rr; *chi2 = x2;
  return true;
}

// P[0..4]: anchors; (k3a, sk3a), (k3b, sk3b): stored kappa3 / sigma of T3 (1,2,3) and (3,4,5).
LST_HD bool t5_eval_d(const Params &g, const Pt *P, double k3a, double sk3a, double k3b, double sk3b, T5Out *o) {
  if (!le(fabs(k3a - k3b), g.ns * (sk3a + sk3b))) return false;              // T5-1 radius match
  if (!t3_eval_d(g, P[1], P[2], P[3], nullptr)) return false;               // T5-2 middle triplet
  if (!(chord_of(P[0], P[2]) > kGuard) || !(chord_of(P[2], P[4]) > kGuard) || !(chord_of(P[0], P[4]) > kGuard))
    return false;
  const double k135 = kappa3_of(P[0], P[2], P[4]);
  double R = 0.0, chi2 = 0.0;
  if (!kasa_fit_d(g, P, fabs(k135), &R, &chi2)) return false;                // T5-3 circle fit
  if (!le(chi2, g.chi2max)) return false;
  const double k5 = (k135 > 0.0 ? 1.0 : (k135 < 0.0 ? -1.0 : 0.0)) / (2.0 * R);
  const double den = arc_of(P[4].rt, k5) - arc_of(P[0].rt, k5);
  if (!(den > kGuard)) return false;
  if (o) {
    o->R = R; o->chi2 = chi2;
    o->pt = g.kB * R;
    o->phi = wrap_pi(atan2(P[0].y, P[0].x) - asin(clamp1(k5 * P[0].rt)));
    o->eta = asinh((P[4].z - P[0].z) / den);
  }
  return true;
}

// ------------------------------------------------------------------ C6 pixel linking
struct Seed { double pt, eta, phi, z0; int q; };

// All n anchors of an OT object against one pixel seed.  first_layer = logical layer of the first MD.
LST_HD bool px_eval_d(const Params &g, const Seed &s, const Pt *P, int n, int first_layer, double *chi2) {
  if (!((g.start_mask >> first_layer) & 1u)) return false;
  if (!(s.pt > kGuard)) return false;
  const double kp = -(double)s.q * g.kB / (2.0 * s.pt);
  const double sh = sinh(s.eta);
  double sum = 0.0;
  for (int k = 0; k < n; ++k) {
    const Pt &h = P[k];
    const bool ec = is_endcap(h.cat);
    double al;
    if (!ec) al = arc_of(h.rt, kp);
    else {
      if (!(fabs(sh) > kGuard)) return false;
      al = (h.z - s.z0) / sh;
    }
    if (!(al > 0.0)) return false;
    const double dph = wrap_pi(atan2(h.y, h.x) - (s.phi + kp * al));
    const double sphi = g.seed_sig_phi + g.seed_sig_pt * fabs(kp) * al + g.sig_t[h.cat] / h.rt;
    double dzt, szt;
    if (!ec) {
      dzt = h.z - (s.z0 + sh * al);
      szt = g.seed_sig_z + g.sig_z[h.cat];
    } else {
      const double rp = (fabs(kp * al) <= 1e-4) ? al : sin(kp * al) / kp;
      dzt = h.rt - rp;
      szt = g.seed_sig_z / fabs(sh) + g.sig_r[h.cat];
    }
    if (!le(fabs(dph), g.ns * sphi)) return false;
    if (!le(fabs(dzt), g.ns * szt)) return false;
    sum += (dph / sphi) * (dph / sphi) + (dzt / szt) * (dzt / szt);
  }
  *chi2 = sum / (2.0 * n);
  return true;
}

}  // namespace lst
