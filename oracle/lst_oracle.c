/* lst_oracle.c -- see lst_oracle.h.  TEST INFRASTRUCTURE ONLY.
 *
 * Notation follows DESIGN.md "Readings of the paper" (C0-C7).  PAPER.md line numbers refer to
 * /root/reference/PAPER.md (arxiv 2209.13711).  Everything is exhaustive enumeration plus
 * predicates; no blocking, no early exit inside a predicate (all cuts are evaluated so that the
 * margin = min_k |v_k - thr_k| / |thr_k| is defined for every candidate).
 */
#include "lst_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define GUARD 1e-9

/* ------------------------------------------------------------------ containers */
typedef struct { double x, y, z, rt; int cat; } pt3;

typedef struct {
  uint32_t hl, hu, module;
  pt3 a;                 /* anchor = lower hit (C0) */
  double kappa, sigk, dphi, margin;
} md_t;
typedef struct { uint32_t mi, mo; double kappa, sigk, dphi, margin; } ls_t;
typedef struct { uint32_t la, lb, m[3]; double kappa3, sigk3, beta, margin; } t3_t;
typedef struct {
  uint32_t ta, tb, m[5];
  double R, chi2, k3a, k3b, pt, eta, phi, margin;
} t5_t;
typedef struct { uint32_t pls, obj; double chi2, margin; } px_t;
typedef struct { uint32_t type, obj; double pt, eta, phi; } tc_t;

#define VEC(T) struct { T *v; uint32_t n, cap; }
#define VPUSH(vec, item) do { \
  if ((vec).n == (vec).cap) { (vec).cap = (vec).cap ? 2 * (vec).cap : 1024; \
    (vec).v = realloc((vec).v, (size_t)(vec).cap * sizeof(*(vec).v)); } \
  (vec).v[(vec).n++] = (item); } while (0)
#define VCLEAR(vec) ((vec).n = 0)
#define VFREE(vec) do { free((vec).v); (vec).v = NULL; (vec).n = (vec).cap = 0; } while (0)

struct lsto_ctx {
  lsto_config cfg;
  double kmax;
  uint32_t n_modules;
  uint8_t *category, *layer;
  uint32_t *map_off, *map_cols;
  /* event */
  uint32_t n_hits, n_seeds;
  double *hx, *hy, *hz;
  uint32_t *hdet;
  uint32_t *det_off, *det_hits;      /* hits grouped by det, ascending original index */
  double *spt, *seta, *sphi, *sz0;
  int8_t *sq;
  uint32_t *sids;
  /* objects */
  VEC(md_t) md;
  VEC(ls_t) ls;
  VEC(t3_t) t3;
  VEC(t5_t) t5;
  VEC(px_t) pt3, pt5;
  VEC(tc_t) tc;
  float *phic;                       /* [n_modules] module centre azimuth: set by lsto_set_truncation (azimuth order) */
  uint32_t trunc[6][16];             /* occupancy caps per level and logical layer (0 = none)                         */
  int s0_fixpoint;                   /* lsto_set_s0_fixpoint: greedy (fix-point) S0 for the T5 collection              */
  uint32_t *md_mod_off;              /* [n_modules+1] MD range of a module          */
  uint32_t *ls_md_off;               /* [n_md+1]      LS range of an inner MD       */
  uint32_t *t3_md_off;               /* [n_md+1]      T3 range of a first MD        */
  uint8_t *keep_t5, *keep_pt3, *keep_pt5, *keep_pls;
};

/* ------------------------------------------------------------------ config */
void lsto_default_config(lsto_config *c) {
  const double s12 = sqrt(12.0);
  memset(c, 0, sizeof(*c));
  c->kB = 0.00299792458 * 3.8;
  c->pt_min = 0.8;
  c->n_sigma = 4.0;
  c->z0max = 15.0;
  c->d0max = 2.5;
  c->chi2max = 18.42;
  c->dr2max = 1e-4;
  c->map_kscale = 1.25;
  c->map_z0 = 20.0;
  c->ec_md_sys = 0.3;
  c->modez_slack = 0.15;
  c->seed_sig_phi = 0.001;
  c->seed_sig_pt = 0.01;
  c->seed_sig_z = 0.05;
  const double st[4] = {0.01, 0.009, 0.01, 0.009}, sz[4] = {0.15, 5.0, 0, 0}, sr[4] = {0, 0, 0.15, 5.0};
  for (int k = 0; k < 4; ++k) { c->sig_t[k] = st[k] / s12; c->sig_z[k] = sz[k] / s12; c->sig_r[k] = sr[k] / s12; }
  c->dup_t5_shared = 5;
  c->dup_pt5_shared = 5;
  c->dup_pt3_shared = 3;
  c->s0_enabled = 1;
  c->start_layer_mask = (1u << 0) | (1u << 1) | (1u << 6) | (1u << 7) | (1u << 11) | (1u << 12);
}

/* ------------------------------------------------------------------ C0 helpers */
static double cross2(double ax, double ay, double bx, double by) { return ax * by - ay * bx; }
static double dot2(double ax, double ay, double bx, double by) { return ax * bx + ay * by; }
static double clamp1(double v) { return v > 1.0 ? 1.0 : (v < -1.0 ? -1.0 : v); }
static double min2(double a, double b) { return a < b ? a : b; }
static double max2(double a, double b) { return a > b ? a : b; }
static double wrap_pi(double a) { return remainder(a, 2.0 * 3.14159265358979323846); }
static int is_endcap(int cat) { return cat >= 2; }

/* sd(A,B) = cross(A, B-A) / (rt_A rt_B) = sin(dphi), difference first (C0) */
static double sd_f(const pt3 *A, const pt3 *B) {
  return cross2(A->x, A->y, B->x - A->x, B->y - A->y) / (A->rt * B->rt);
}
static double dphi_f(const pt3 *A, const pt3 *B) {
  return atan2(cross2(A->x, A->y, B->x - A->x, B->y - A->y), dot2(A->x, A->y, B->x, B->y));
}
static double chord_f(const pt3 *A, const pt3 *B) { return hypot(B->x - A->x, B->y - A->y); }
/* dr(A,B) = rt_B - rt_A without cancellation (C0) */
static double dr_f(const pt3 *A, const pt3 *B) {
  double dx = B->x - A->x, dy = B->y - A->y;
  return (2.0 * dot2(A->x, A->y, dx, dy) + dot2(dx, dy, dx, dy)) / (A->rt + B->rt);
}
/* three-point half curvature (Menger / 2), C0 */
static double kappa3_f(const pt3 *A, const pt3 *B, const pt3 *C) {
  double abx = B->x - A->x, aby = B->y - A->y, bcx = C->x - B->x, bcy = C->y - B->y;
  double acx = C->x - A->x, acy = C->y - A->y;
  return cross2(abx, aby, bcx, bcy) / (hypot(abx, aby) * hypot(bcx, bcy) * hypot(acx, acy));
}
/* arc length at transverse distance r on a prompt circle of half curvature k (C0) */
static double arc_f(double r, double k) {
  if (fabs(k * r) <= 1e-4) return r;
  return asin(clamp1(k * r)) / k;
}

/* cut bookkeeping: pass &= (v <= thr) (NaN fails); margin = min |v-thr|/|thr| */
typedef struct { int pass; double margin; } cut_t;
/* test hook (lsto_test_cuts): while a trace buffer is installed every cut appends the triple
 * (kind, v, thr) in evaluation order; kind 0 = "v <= thr", 1 = "v > 0" (thr = its scale),
 * 2 = a guard failed (v = thr = 0).  It records the bookkeeping, it changes no arithmetic. */
static _Thread_local double *g_trace = NULL;
static _Thread_local int g_trace_n = 0, g_trace_cap = 0;
static void trace_push(double kind, double v, double thr) {
  if (g_trace && g_trace_n + 3 <= g_trace_cap) {
    g_trace[g_trace_n] = kind; g_trace[g_trace_n + 1] = v; g_trace[g_trace_n + 2] = thr;
  }
  if (g_trace) g_trace_n += 3;
}
static void cut_le(cut_t *c, double v, double thr) {
  trace_push(0.0, v, thr);
  if (!(v <= thr)) c->pass = 0;
  double m = fabs(v - thr) / max2(fabs(thr), 1e-300);
  if (!(m >= 0.0)) m = 0.0; /* NaN: treat as on-threshold */
  if (m < c->margin) c->margin = m;
}
/* sign requirement v > 0, measured against a natural scale */
static void cut_pos(cut_t *c, double v, double scale) {
  trace_push(1.0, v, scale);
  if (!(v > 0.0)) c->pass = 0;
  double m = fabs(v) / max2(fabs(scale), 1e-300);
  if (!(m >= 0.0)) m = 0.0;
  if (m < c->margin) c->margin = m;
}
static void cut_fail(cut_t *c) { trace_push(2.0, 0.0, 0.0); c->pass = 0; }

/* ------------------------------------------------------------------ C1 mini-doublets
 * PAPER.md:37 (Fig. 2): a stub is a pair of hits in the two sensors of one pT module inside a
 * window equivalent to pT >= 0.8 GeV. */
static cut_t md_eval(const lsto_ctx *c, const pt3 *l, const pt3 *u, int cat, md_t *out) {
  const lsto_config *g = &c->cfg;
  cut_t r = {1, INFINITY};
  if (!(l->rt > GUARD) || !(u->rt > GUARD)) { cut_fail(&r); return r; }
  double dz = u->z - l->z;
  double sdv = sd_f(l, u), cxy = chord_f(l, u), drv = dr_f(l, u);
  double st = g->sig_t[cat];
  double tolphi = g->n_sigma * st * (1.0 / l->rt + 1.0 / u->rt);
  double cpred;
  if (!is_endcap(cat)) {
    /* B1: pointing in r-z */
    cut_pos(&r, drv, l->rt);
    cut_le(&r, fabs(dz - l->z * drv / l->rt), g->z0max * drv / l->rt + 2.0 * g->n_sigma * g->sig_z[cat]);
    /* B2: pT window */
    cut_le(&r, fabs(sdv), c->kmax * cxy + tolphi);
    cpred = cxy;
  } else {
    double azl = fabs(l->z);
    if (!(azl > GUARD) || !(azl - g->z0max > GUARD)) { cut_fail(&r); return r; }
    /* E1 */
    cut_le(&r, fabs(drv - l->rt * dz / l->z),
           l->rt * fabs(dz) * g->z0max / (azl * (azl - g->z0max)) + 2.0 * g->n_sigma * g->sig_r[cat]);
    /* E2 */
    cut_le(&r, fabs(sdv), fabs(dz) * asin(min2(1.0, c->kmax * l->rt)) / (azl - g->z0max) + tolphi);
    cpred = fabs(dz) * l->rt / azl;
  }
  if (!(cpred > GUARD)) { cut_fail(&r); return r; }
  if (out) {
    out->a = *l;
    out->a.cat = cat;
    out->kappa = sdv / cpred;
    out->sigk = st * (1.0 / l->rt + 1.0 / u->rt) / cpred;
    out->dphi = asin(clamp1(sdv));
    out->margin = r.margin;
  }
  return r;
}

/* ------------------------------------------------------------------ C3 line segments
 * PAPER.md:53-55 (Fig. 4-7): stubs in neighbouring layers, module-map pairs only, geometric cuts. */
static cut_t ls_eval(const lsto_ctx *c, const md_t *i, const md_t *o, ls_t *out) {
  const lsto_config *g = &c->cfg;
  cut_t r = {1, INFINITY};
  const pt3 *A = &i->a, *B = &o->a;
  int ci = A->cat, co = B->cat;
  int modeZ = is_endcap(co);
  double ns = g->n_sigma;
  double dz = B->z - A->z;
  double drv = dr_f(A, B), sdv = sd_f(A, B), cxy = chord_f(A, B), dph = dphi_f(A, B);
  /* L1 pointing: origin-to-line distance in r-z, no division */
  double N = A->rt * dz - A->z * drv;
  double E = A->rt * g->sig_z[co] + B->rt * g->sig_z[ci] + fabs(B->z) * g->sig_r[ci] + fabs(A->z) * g->sig_r[co];
  cut_le(&r, fabs(N), g->z0max * fabs(drv) + ns * E);
  /* L2 pT window */
  double tphi = g->sig_t[ci] / A->rt + g->sig_t[co] / B->rt;
  double tolphi = ns * tphi;
  cut_pos(&r, dot2(A->x, A->y, B->x, B->y), A->rt * B->rt);
  double kls, sigkls, slack;
  if (!modeZ) {
    if (!(cxy > GUARD)) { cut_fail(&r); return r; }
    cut_le(&r, fabs(sdv), c->kmax * cxy + tolphi);
    kls = sdv / cxy;
    sigkls = tphi / cxy;
    slack = 0.0;
  } else {
    double rbar = 0.5 * (A->rt + B->rt), zbar = 0.5 * (fabs(A->z) + fabs(B->z));
    double adz = fabs(dz);
    if (!(adz > GUARD) || !(rbar > GUARD)) { cut_fail(&r); return r; }
    double Sbar = asin(min2(1.0, c->kmax * (rbar + ns * (g->sig_r[ci] + g->sig_r[co]) / 2.0))) / c->kmax;
    double den = zbar - g->z0max - ns * g->sig_z[ci] / 2.0;
    cut_pos(&r, den, zbar);
    if (!(den > GUARD)) { cut_fail(&r); return r; }
    cut_le(&r, fabs(dph), c->kmax * (adz + ns * g->sig_z[ci]) * Sbar / den + tolphi);
    double lever = zbar / (adz * rbar);
    kls = dph * lever;
    sigkls = tphi * lever;
    slack = fabs(kls) * (g->z0max / zbar + g->modez_slack + ns * (g->sig_r[ci] + g->sig_r[co]) / (A->rt + B->rt) +
                         ns * g->sig_z[ci] / adz);
  }
  /* L3 stub-segment curvature consistency */
  cut_le(&r, fabs(i->kappa - kls), ns * (i->sigk + sigkls) + slack + (is_endcap(ci) ? g->ec_md_sys * fabs(kls) : 0.0));
  cut_le(&r, fabs(o->kappa - kls), ns * (o->sigk + sigkls) + slack + (is_endcap(co) ? g->ec_md_sys * fabs(kls) : 0.0));
  if (out) { out->kappa = kls; out->sigk = sigkls; out->dphi = dph; out->margin = r.margin; }
  return r;
}

/* ------------------------------------------------------------------ C4 triplets
 * PAPER.md:73 (Fig. 5, 8): two segments sharing a stub; the relative angle between the segments
 * rejects unphysical patterns. */
static double sig_perp(const lsto_ctx *c, const pt3 *h) {
  return c->cfg.sig_t[h->cat] + c->cfg.sig_r[h->cat] * min2(1.0, c->kmax * h->rt);
}
static cut_t t3_eval(const lsto_ctx *c, const pt3 *P1, const pt3 *P2, const pt3 *P3, t3_t *out) {
  const lsto_config *g = &c->cfg;
  cut_t r = {1, INFINITY};
  double ns = g->n_sigma;
  int modeZ = is_endcap(P1->cat) || is_endcap(P2->cat) || is_endcap(P3->cat);
  double d12x = P2->x - P1->x, d12y = P2->y - P1->y, d23x = P3->x - P2->x, d23y = P3->y - P2->y;
  double a = hypot(d12x, d12y), b = hypot(d23x, d23y), c13 = chord_f(P1, P3);
  if (!(a > GUARD) || !(b > GUARD) || !(c13 > GUARD)) { cut_fail(&r); return r; }
  /* T3-1 relative angle (beta) cut */
  double k3 = kappa3_f(P1, P2, P3);
  double sk3 = (sig_perp(c, P2) + (b * sig_perp(c, P1) + a * sig_perp(c, P3)) / c13) / (a * b);
  cut_le(&r, fabs(k3), c->kmax + ns * sk3);
  double beta = atan2(cross2(d12x, d12y, d23x, d23y), dot2(d12x, d12y, d23x, d23y));
  /* T3-2 phi-lever linearity */
  double d12 = dphi_f(P1, P2), d23 = dphi_f(P2, P3), d13 = d12 + d23;
  double k13 = sin(d13) / c13;
  double L1, L2, L3, sL1, sL2, sL3;
  if (modeZ) {
    L1 = P1->z; L2 = P2->z; L3 = P3->z;
    sL1 = g->sig_z[P1->cat]; sL2 = g->sig_z[P2->cat]; sL3 = g->sig_z[P3->cat];
  } else {
    L1 = arc_f(P1->rt, k13); L2 = arc_f(P2->rt, k13); L3 = arc_f(P3->rt, k13);
    sL1 = sL2 = sL3 = 0.0;
  }
  double Nphi = d12 * (L3 - L2) - d23 * (L2 - L1);
  double Nrho = (1.0 / P2->rt - 1.0 / P1->rt) * (L3 - L2) - (1.0 / P3->rt - 1.0 / P2->rt) * (L2 - L1);
  double Ephi = g->sig_t[P1->cat] / P1->rt * fabs(L3 - L2) + g->sig_t[P2->cat] / P2->rt * fabs(L3 - L1) +
                g->sig_t[P3->cat] / P3->rt * fabs(L2 - L1) + sL1 * fabs(d23) + sL2 * fabs(d13) + sL3 * fabs(d12);
  cut_le(&r, fabs(Nphi), g->d0max * fabs(Nrho) + ns * Ephi);
  /* T3-3 r-z collinearity */
  double s1 = P1->rt * (1.0 + (k3 * P1->rt) * (k3 * P1->rt) / 6.0);
  double s2 = P2->rt * (1.0 + (k3 * P2->rt) * (k3 * P2->rt) / 6.0);
  double s3 = P3->rt * (1.0 + (k3 * P3->rt) * (k3 * P3->rt) / 6.0);
  double Nz = (s2 - s1) * (P3->z - P1->z) - (s3 - s1) * (P2->z - P1->z);
  double Ez = g->sig_z[P3->cat] * fabs(s2 - s1) + g->sig_z[P2->cat] * fabs(s3 - s1) + g->sig_z[P1->cat] * fabs(s3 - s2) +
              g->sig_r[P2->cat] * fabs(P3->z - P1->z) + g->sig_r[P3->cat] * fabs(P2->z - P1->z) +
              g->sig_r[P1->cat] * fabs(P3->z - P2->z);
  cut_le(&r, fabs(Nz), ns * Ez);
  if (out) { out->kappa3 = k3; out->sigk3 = sk3; out->beta = beta; out->margin = r.margin; }
  return r;
}

/* ------------------------------------------------------------------ C5 quintuplets
 * PAPER.md:73 (Fig. 9): two triplets sharing a stub; north_star: circle-fit chi2 cut. */
static int kasa_fit(const lsto_ctx *c, const pt3 *P[5], double kc, double *R, double *chi2, double *detn) {
  double w[5], sw = 0, mx = 0, my = 0;
  for (int k = 0; k < 5; ++k) {
    double st = c->cfg.sig_t[P[k]->cat], sr = c->cfg.sig_r[P[k]->cat] * min2(1.0, kc * P[k]->rt);
    w[k] = 1.0 / (st * st + sr * sr);
    sw += w[k]; mx += w[k] * P[k]->x; my += w[k] * P[k]->y;
  }
  mx /= sw; my /= sw;
  double u[5], v[5], Suu = 0, Suv = 0, Svv = 0, Suz = 0, Svz = 0, Sz = 0;
  for (int k = 0; k < 5; ++k) {
    u[k] = P[k]->x - mx; v[k] = P[k]->y - my;
    double zeta = u[k] * u[k] + v[k] * v[k];
    Suu += w[k] * u[k] * u[k]; Suv += w[k] * u[k] * v[k]; Svv += w[k] * v[k] * v[k];
    Suz += w[k] * u[k] * zeta; Svz += w[k] * v[k] * zeta; Sz += w[k] * zeta;
  }
  double det = Suu * Svv - Suv * Suv;
  *detn = det / max2(Suu * Svv, 1e-300);
  if (!(det > 0.0)) return 0;
  double Bc = (-Suz * Svv + Svz * Suv) / det;
  double Cc = (-Svz * Suu + Suz * Suv) / det;
  double cx = -Bc / 2.0, cy = -Cc / 2.0;
  double R2 = (Bc * Bc + Cc * Cc) / 4.0 + Sz / sw;
  if (!(R2 > 0.0)) return 0;
  *R = sqrt(R2);
  double x2 = 0;
  for (int k = 0; k < 5; ++k) {
    double e = hypot(u[k] - cx, v[k] - cy) - *R;
    x2 += w[k] * e * e;
  }
  *chi2 = x2;
  return 1;
}

static cut_t t5_eval(const lsto_ctx *c, const pt3 *P[5], double k3a, double sk3a, double k3b, double sk3b,
                     t5_t *out) {
  const lsto_config *g = &c->cfg;
  cut_t r = {1, INFINITY};
  /* T5-1 radius match */
  cut_le(&r, fabs(k3a - k3b), g->n_sigma * (sk3a + sk3b));
  /* T5-2 middle triplet */
  cut_t mid = t3_eval(c, P[1], P[2], P[3], NULL);
  if (!mid.pass) r.pass = 0;
  if (mid.margin < r.margin) r.margin = mid.margin;
  /* T5-3 circle fit */
  if (!(chord_f(P[0], P[2]) > GUARD) || !(chord_f(P[2], P[4]) > GUARD) || !(chord_f(P[0], P[4]) > GUARD)) {
    cut_fail(&r); return r;
  }
  double k135 = kappa3_f(P[0], P[2], P[4]);
  double R = 0, chi2 = 0, detn = 0;
  int ok = kasa_fit(c, P, fabs(k135), &R, &chi2, &detn);
  cut_pos(&r, detn, 1.0);
  if (!ok) { cut_fail(&r); return r; }
  cut_le(&r, chi2, g->chi2max);
  double k5 = (k135 > 0 ? 1.0 : (k135 < 0 ? -1.0 : 0.0)) / (2.0 * R);
  double den = arc_f(P[4]->rt, k5) - arc_f(P[0]->rt, k5);
  cut_pos(&r, den - GUARD, P[4]->rt);
  if (!(den > GUARD)) { cut_fail(&r); return r; }
  if (out) {
    out->R = R; out->chi2 = chi2; out->k3a = k3a; out->k3b = k3b;
    out->pt = g->kB * R;
    out->phi = wrap_pi(atan2(P[0]->y, P[0]->x) - asin(clamp1(k5 * P[0]->rt)));
    out->eta = asinh((P[4]->z - P[0]->z) / den);
    out->margin = r.margin;
  }
  return r;
}

/* ------------------------------------------------------------------ C6 pixel linking
 * PAPER.md:75 (Fig. 10-11): T3 / T5 linked to a pixel line segment. */
/* full = 0: the bulk enumeration stops at the first failing anchor (same pass/fail; the margin of a
 * passing pair still covers all anchors).  full = 1 (lsto_eval): every cut of every anchor. */
static cut_t px_eval(const lsto_ctx *c, uint32_t p, const pt3 *const *P, int n, int first_layer, double *chi2,
                     int full) {
  const lsto_config *g = &c->cfg;
  cut_t r = {1, INFINITY};
  if (!((g->start_layer_mask >> first_layer) & 1u)) { cut_fail(&r); return r; }
  double pt = c->spt[p], eta = c->seta[p], phi = c->sphi[p], z0 = c->sz0[p];
  if (!(pt > GUARD)) { cut_fail(&r); return r; }
  double kp = -(double)c->sq[p] * g->kB / (2.0 * pt);
  double sh = sinh(eta);
  double sum = 0;
  for (int k = 0; k < n; ++k) {
    const pt3 *h = P[k];
    double s;
    int ec = is_endcap(h->cat);
    if (!ec) s = arc_f(h->rt, kp);
    else {
      if (!(fabs(sh) > GUARD)) { cut_fail(&r); return r; }
      s = (h->z - z0) / sh;
    }
    cut_pos(&r, s, h->rt);
    double dph = wrap_pi(atan2(h->y, h->x) - (phi + kp * s));
    double sphi = g->seed_sig_phi + g->seed_sig_pt * fabs(kp) * s + g->sig_t[h->cat] / h->rt;
    double dzt, szt;
    if (!ec) {
      dzt = h->z - (z0 + sh * s);
      szt = g->seed_sig_z + g->sig_z[h->cat];
    } else {
      double rp = (fabs(kp * s) <= 1e-4) ? s : sin(kp * s) / kp;
      dzt = h->rt - rp;
      szt = g->seed_sig_z / fabs(sh) + g->sig_r[h->cat];
    }
    cut_le(&r, fabs(dph), g->n_sigma * sphi);
    cut_le(&r, fabs(dzt), g->n_sigma * szt);
    if (!full && !r.pass) return r;
    sum += (dph / sphi) * (dph / sphi) + (dzt / szt) * (dzt / szt);
  }
  *chi2 = sum / (2.0 * n);
  return r;
}

/* ------------------------------------------------------------------ C2 module map
 * PAPER.md:53-55 (Fig. 4): modules reachable from a reference module by +- helices from the
 * detector centre at the pT threshold.  Deterministic interval version (reading C2). */
static int next_layers(int L, int out[3]) {
  int n = 0;
  if (L < 6) { if (L + 1 < 6) out[n++] = L + 1; out[n++] = 6; out[n++] = 11; }
  else if ((L >= 6 && L < 10) || (L >= 11 && L < 15)) out[n++] = L + 1;
  return n;
}
static int map_connected(const lsto_config *g, double kp, int ecB, double rminA, double rmaxA, double phiA,
                         double hpA, double zminA, double zmaxA, double rminB, double rmaxB, double phiB,
                         double hpB, double zminB, double zmaxB) {
  double aA = asin(min2(1.0, kp * rminA)), aB = asin(min2(1.0, kp * rmaxB));
  double dphi = fabs(wrap_pi(phiB - phiA));
  if (!(dphi <= hpA + hpB + aB - aA + g->d0max * max2(0.0, 1.0 / rminA - 1.0 / rmaxB))) return 0;
  double rho_lo = rminB / rmaxA, rho_hi = aB / aA;
  double z0s[2] = {-g->map_z0, g->map_z0}, zAs[2] = {zminA, zmaxA}, rhos[2] = {rho_lo, rho_hi};
  if (!ecB) {
    double lo = INFINITY, hi = -INFINITY;
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) for (int k = 0; k < 2; ++k) {
      double zp = z0s[a] + (zAs[b] - z0s[a]) * rhos[k];
      lo = min2(lo, zp); hi = max2(hi, zp);
    }
    return (lo <= zmaxB) && (hi >= zminB);
  } else {
    double side = zminB > 0 ? 1.0 : -1.0, zB = zminB;
    double lo = INFINITY, hi = -INFINITY;
    int nvalid = 0;
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) {
      double den = zAs[b] - z0s[a];
      if (!(side * den > 0.0)) continue;
      double q = (zB - z0s[a]) / den;
      lo = min2(lo, q); hi = max2(hi, q);
      ++nvalid;
    }
    if (nvalid == 0) return 0;
    if (nvalid < 4) hi = INFINITY; /* the ratio is unbounded where z_A - z0 -> 0 */
    return (lo <= rho_hi) && (hi >= rho_lo);
  }
}
int lsto_build_module_map(uint32_t n, const uint8_t *category, const uint8_t *layer, const float *rmin,
                          const float *rmax, const float *phic, const float *half_phi, const float *zmin,
                          const float *zmax, const lsto_config *g, uint32_t **row_offsets, uint32_t **cols) {
  double kp = g->map_kscale * g->kB / (2.0 * g->pt_min);
  uint32_t *off = calloc((size_t)n + 1, sizeof(uint32_t));
  VEC(uint32_t) cv = {0};
  for (uint32_t A = 0; A < n; ++A) {
    int nl[3], nn = next_layers(layer[A], nl);
    off[A] = cv.n;
    for (uint32_t B = 0; B < n; ++B) {
      int ok = 0;
      for (int k = 0; k < nn; ++k) if (layer[B] == nl[k]) ok = 1;
      if (!ok) continue;
      if (map_connected(g, kp, category[B] >= 2, rmin[A], rmax[A], phic[A], half_phi[A], zmin[A], zmax[A],
                        rmin[B], rmax[B], phic[B], half_phi[B], zmin[B], zmax[B]))
        VPUSH(cv, B);
    }
  }
  off[n] = cv.n;
  if (!cv.v) cv.v = malloc(sizeof(uint32_t));
  *row_offsets = off;
  *cols = cv.v;
  return 0;
}
void lsto_free(void *p) { free(p); }

/* ------------------------------------------------------------------ context / event */
lsto_ctx *lsto_create(uint32_t n_modules, const uint8_t *category, const uint8_t *layer,
                      const uint32_t *map_offsets, const uint32_t *map_cols, const lsto_config *cfg) {
  lsto_ctx *c = calloc(1, sizeof(*c));
  if (cfg) c->cfg = *cfg; else lsto_default_config(&c->cfg);
  c->kmax = c->cfg.kB / (2.0 * c->cfg.pt_min);
  c->n_modules = n_modules;
  c->category = malloc(n_modules); memcpy(c->category, category, n_modules);
  c->layer = malloc(n_modules); memcpy(c->layer, layer, n_modules);
  c->map_off = malloc(((size_t)n_modules + 1) * 4); memcpy(c->map_off, map_offsets, ((size_t)n_modules + 1) * 4);
  uint32_t ne = map_offsets[n_modules];
  c->map_cols = malloc(((size_t)ne + 1) * 4); memcpy(c->map_cols, map_cols, (size_t)ne * 4);
  return c;
}
static void free_event(lsto_ctx *c) {
  free(c->hx); free(c->hy); free(c->hz); free(c->hdet); free(c->det_off); free(c->det_hits);
  free(c->spt); free(c->seta); free(c->sphi); free(c->sz0); free(c->sq); free(c->sids);
  c->hx = c->hy = c->hz = NULL; c->hdet = c->det_off = c->det_hits = NULL;
  c->spt = c->seta = c->sphi = c->sz0 = NULL; c->sq = NULL; c->sids = NULL;
  VCLEAR(c->md); VCLEAR(c->ls); VCLEAR(c->t3); VCLEAR(c->t5); VCLEAR(c->pt3); VCLEAR(c->pt5); VCLEAR(c->tc);
  free(c->md_mod_off); free(c->ls_md_off); free(c->t3_md_off);
  c->md_mod_off = c->ls_md_off = c->t3_md_off = NULL;
  free(c->keep_t5); free(c->keep_pt3); free(c->keep_pt5); free(c->keep_pls);
  c->keep_t5 = c->keep_pt3 = c->keep_pt5 = c->keep_pls = NULL;
}
void lsto_destroy(lsto_ctx *c) {
  if (!c) return;
  free_event(c);
  VFREE(c->md); VFREE(c->ls); VFREE(c->t3); VFREE(c->t5); VFREE(c->pt3); VFREE(c->pt5); VFREE(c->tc);
  free(c->category); free(c->layer); free(c->map_off); free(c->map_cols); free(c->phic);
  free(c);
}

/* PAPER.md:125 (occupancy truncation).  Optional mode: a bucket (MD, LS, T3, T5: the
 * module of the object's first MD; pT3 / pT5: the pixel seed) keeps at most K objects, the K FIRST in
 * the enumeration order of the definition, where the hits of a sensor are taken in ascending azimuth
 * relative to the module centre phic (ties: original index).  caps: 6 x 16 values, level-major (MD,
 * LS, T3, T5, PT3, PT5) by logical layer of the bucket's module (pixel levels: entry 0), 0 = no cap.
 * Must be called before lsto_load_event.  The all-pairs (brute) builders ignore the caps. */
int lsto_set_truncation(lsto_ctx *c, const float *phic, const uint32_t *caps) {
  if (!c || !phic) return -1;
  free(c->phic);
  c->phic = malloc(((size_t)c->n_modules + 1) * sizeof(float));
  memcpy(c->phic, phic, (size_t)c->n_modules * sizeof(float));
  memset(c->trunc, 0, sizeof(c->trunc));
  if (caps) memcpy(c->trunc, caps, sizeof(c->trunc));
  return 0;
}
static uint32_t trunc_cap(const lsto_ctx *c, int level, uint32_t module) { return c->trunc[level][c->layer[module] & 15]; }

int lsto_load_event(lsto_ctx *c, uint32_t n_hits, const float *x, const float *y, const float *z,
                    const uint32_t *det, uint32_t n_seeds, const float *pt, const float *eta,
                    const float *phi, const float *z0, const int8_t *q, const uint32_t *hit_ids) {
  free_event(c);
  for (uint32_t h = 0; h < n_hits; ++h)
    if (det[h] >= 2 * c->n_modules) return -1;
  c->n_hits = n_hits; c->n_seeds = n_seeds;
  c->hx = malloc(((size_t)n_hits + 1) * 8); c->hy = malloc(((size_t)n_hits + 1) * 8);
  c->hz = malloc(((size_t)n_hits + 1) * 8); c->hdet = malloc(((size_t)n_hits + 1) * 4);
  for (uint32_t h = 0; h < n_hits; ++h) { c->hx[h] = x[h]; c->hy[h] = y[h]; c->hz[h] = z[h]; c->hdet[h] = det[h]; }
  /* group hits by det, ascending original index inside a det */
  uint32_t nd = 2 * c->n_modules;
  c->det_off = calloc((size_t)nd + 1, 4);
  c->det_hits = malloc(((size_t)n_hits + 1) * 4);
  for (uint32_t h = 0; h < n_hits; ++h) c->det_off[det[h] + 1]++;
  for (uint32_t d = 0; d < nd; ++d) c->det_off[d + 1] += c->det_off[d];
  uint32_t *fill = malloc(((size_t)nd + 1) * 4);
  memcpy(fill, c->det_off, ((size_t)nd + 1) * 4);
  for (uint32_t h = 0; h < n_hits; ++h) c->det_hits[fill[det[h]]++] = h;
  free(fill);
  if (c->phic) {
    /* occupancy-truncation mode (lsto_set_truncation): inside a det the hits ascend in azimuth relative
     * to the module centre (ties: original index), so that every level is enumerated in the order the
     * truncation rule "keep the first K of a bucket" refers to.  Insertion sort: a det holds ~10 hits. */
    for (uint32_t d = 0; d < nd; ++d) {
      uint32_t a = c->det_off[d], b = c->det_off[d + 1];
      for (uint32_t i = a + 1; i < b; ++i) {
        uint32_t h = c->det_hits[i];
        double kh = wrap_pi(atan2(c->hy[h], c->hx[h]) - (double)c->phic[d >> 1]);
        uint32_t j = i;
        while (j > a) {
          uint32_t g = c->det_hits[j - 1];
          double kg = wrap_pi(atan2(c->hy[g], c->hx[g]) - (double)c->phic[d >> 1]);
          if (kg < kh || (kg == kh && g < h)) break;
          c->det_hits[j] = g; --j;
        }
        c->det_hits[j] = h;
      }
    }
  }
  c->spt = malloc(((size_t)n_seeds + 1) * 8); c->seta = malloc(((size_t)n_seeds + 1) * 8);
  c->sphi = malloc(((size_t)n_seeds + 1) * 8); c->sz0 = malloc(((size_t)n_seeds + 1) * 8);
  c->sq = malloc((size_t)n_seeds + 1); c->sids = malloc(((size_t)n_seeds + 1) * 16);
  for (uint32_t s = 0; s < n_seeds; ++s) {
    c->spt[s] = pt[s]; c->seta[s] = eta[s]; c->sphi[s] = phi[s]; c->sz0[s] = z0[s]; c->sq[s] = q[s];
    for (int k = 0; k < 4; ++k) c->sids[4 * s + k] = hit_ids[4 * s + k];
  }
  return 0;
}

static pt3 hit_pt(const lsto_ctx *c, uint32_t h, int cat) {
  pt3 p = {c->hx[h], c->hy[h], c->hz[h], 0.0, cat};
  p.rt = sqrt(p.x * p.x + p.y * p.y);
  return p;
}

/* ------------------------------------------------------------------ stages */
int lsto_build_md(lsto_ctx *c) {
  VCLEAR(c->md);
  free(c->md_mod_off);
  c->md_mod_off = calloc((size_t)c->n_modules + 1, 4);
  for (uint32_t m = 0; m < c->n_modules; ++m) {
    c->md_mod_off[m] = c->md.n;
    int cat = c->category[m];
    for (uint32_t a = c->det_off[2 * m]; a < c->det_off[2 * m + 1]; ++a) {
      uint32_t hl = c->det_hits[a];
      pt3 l = hit_pt(c, hl, cat);
      for (uint32_t b = c->det_off[2 * m + 1]; b < c->det_off[2 * m + 2]; ++b) {
        uint32_t hu = c->det_hits[b];
        pt3 u = hit_pt(c, hu, cat);
        md_t md; memset(&md, 0, sizeof(md));
        cut_t r = md_eval(c, &l, &u, cat, &md);
        uint32_t K = trunc_cap(c, LSTO_MD, m);
        if (r.pass && !(K && c->md.n - c->md_mod_off[m] >= K)) { md.hl = hl; md.hu = hu; md.module = m; VPUSH(c->md, md); }
      }
    }
  }
  c->md_mod_off[c->n_modules] = c->md.n;
  return 0;
}

static int map_has(const lsto_ctx *c, uint32_t A, uint32_t B) {
  for (uint32_t e = c->map_off[A]; e < c->map_off[A + 1]; ++e) if (c->map_cols[e] == B) return 1;
  return 0;
}

int lsto_build_ls(lsto_ctx *c, int brute) {
  VCLEAR(c->ls);
  free(c->ls_md_off);
  c->ls_md_off = calloc((size_t)c->md.n + 1, 4);
  uint32_t bucket = 0xFFFFFFFFu, in_bucket = 0;     /* occupancy truncation: LS kept so far in the inner MD's module */
  for (uint32_t i = 0; i < c->md.n; ++i) {
    c->ls_md_off[i] = c->ls.n;
    const md_t *mi = &c->md.v[i];
    if (mi->module != bucket) { bucket = mi->module; in_bucket = 0; }
    const uint32_t K = trunc_cap(c, LSTO_LS, mi->module);
    if (brute) {
      for (uint32_t o = 0; o < c->md.n; ++o) {
        const md_t *mo = &c->md.v[o];
        if (!map_has(c, mi->module, mo->module)) continue;
        ls_t ls; memset(&ls, 0, sizeof(ls));
        if (ls_eval(c, mi, mo, &ls).pass) { ls.mi = i; ls.mo = o; VPUSH(c->ls, ls); }
      }
    } else {
      for (uint32_t e = c->map_off[mi->module]; e < c->map_off[mi->module + 1]; ++e) {
        uint32_t B = c->map_cols[e];
        for (uint32_t o = c->md_mod_off[B]; o < c->md_mod_off[B + 1]; ++o) {
          ls_t ls; memset(&ls, 0, sizeof(ls));
          if (ls_eval(c, mi, &c->md.v[o], &ls).pass && !(K && in_bucket >= K)) { ls.mi = i; ls.mo = o; VPUSH(c->ls, ls); ++in_bucket; }
        }
      }
    }
  }
  c->ls_md_off[c->md.n] = c->ls.n;
  return 0;
}

int lsto_build_t3(lsto_ctx *c, int brute) {
  VCLEAR(c->t3);
  free(c->t3_md_off);
  c->t3_md_off = calloc((size_t)c->md.n + 2, 4);
  uint32_t cur_md = 0;
  uint32_t bucket = 0xFFFFFFFFu, in_bucket = 0;     /* occupancy truncation: T3 kept so far in the first MD's module */
  for (uint32_t a = 0; a < c->ls.n; ++a) {
    const ls_t *A = &c->ls.v[a];
    const uint32_t modA = c->md.v[A->mi].module, K = brute ? 0 : trunc_cap(c, LSTO_T3, modA);
    if (modA != bucket) { bucket = modA; in_bucket = 0; }
    while (cur_md <= A->mi) c->t3_md_off[cur_md++] = c->t3.n;   /* T3 are grouped by first MD */
    uint32_t b0 = brute ? 0 : c->ls_md_off[A->mo], b1 = brute ? c->ls.n : c->ls_md_off[A->mo + 1];
    for (uint32_t b = b0; b < b1; ++b) {
      const ls_t *Bq = &c->ls.v[b];
      if (Bq->mi != A->mo) continue;
      t3_t t; memset(&t, 0, sizeof(t));
      const md_t *m1 = &c->md.v[A->mi], *m2 = &c->md.v[A->mo], *m3 = &c->md.v[Bq->mo];
      if (t3_eval(c, &m1->a, &m2->a, &m3->a, &t).pass && !(K && in_bucket >= K)) {
        t.la = a; t.lb = b; t.m[0] = A->mi; t.m[1] = A->mo; t.m[2] = Bq->mo;
        VPUSH(c->t3, t); ++in_bucket;
      }
    }
  }
  while (cur_md <= c->md.n) c->t3_md_off[cur_md++] = c->t3.n;
  return 0;
}

int lsto_build_t5(lsto_ctx *c, int brute) {
  VCLEAR(c->t5);
  uint32_t bucket = 0xFFFFFFFFu, in_bucket = 0;     /* occupancy truncation: T5 kept so far in the first MD's module */
  for (uint32_t a = 0; a < c->t3.n; ++a) {
    const t3_t *A = &c->t3.v[a];
    const uint32_t modA = c->md.v[A->m[0]].module, K = brute ? 0 : trunc_cap(c, LSTO_T5, modA);
    if (modA != bucket) { bucket = modA; in_bucket = 0; }
    uint32_t b0 = brute ? 0 : c->t3_md_off[A->m[2]], b1 = brute ? c->t3.n : c->t3_md_off[A->m[2] + 1];
    for (uint32_t b = b0; b < b1; ++b) {
      const t3_t *Bq = &c->t3.v[b];
      if (Bq->m[0] != A->m[2]) continue;
      uint32_t mm[5] = {A->m[0], A->m[1], A->m[2], Bq->m[1], Bq->m[2]};
      const pt3 *P[5];
      for (int k = 0; k < 5; ++k) P[k] = &c->md.v[mm[k]].a;
      t5_t t; memset(&t, 0, sizeof(t));
      if (t5_eval(c, P, A->kappa3, A->sigk3, Bq->kappa3, Bq->sigk3, &t).pass && !(K && in_bucket >= K)) {
        t.ta = a; t.tb = b;
        for (int k = 0; k < 5; ++k) t.m[k] = mm[k];
        VPUSH(c->t5, t); ++in_bucket;
      }
    }
  }
  return 0;
}

int lsto_link_pixel(lsto_ctx *c, uint32_t s0, uint32_t s1) {
  VCLEAR(c->pt5); VCLEAR(c->pt3);
  if (s1 > c->n_seeds) s1 = c->n_seeds;
  const uint32_t K5 = c->trunc[LSTO_PT5][0], K3 = c->trunc[LSTO_PT3][0];   /* occupancy truncation: per pixel seed */
  for (uint32_t p = s0; p < s1; ++p) {
    uint32_t kept = 0;
    for (uint32_t o = 0; o < c->t5.n; ++o) {
      const t5_t *T = &c->t5.v[o];
      const pt3 *P[5];
      for (int k = 0; k < 5; ++k) P[k] = &c->md.v[T->m[k]].a;
      double chi2 = 0;
      cut_t r = px_eval(c, p, P, 5, c->layer[c->md.v[T->m[0]].module], &chi2, 0);
      if (r.pass && !(K5 && kept >= K5)) { px_t x = {p, o, chi2, r.margin}; VPUSH(c->pt5, x); ++kept; }
    }
  }
  for (uint32_t p = s0; p < s1; ++p) {
    uint32_t kept = 0;
    for (uint32_t o = 0; o < c->t3.n; ++o) {
      const t3_t *T = &c->t3.v[o];
      const pt3 *P[3];
      for (int k = 0; k < 3; ++k) P[k] = &c->md.v[T->m[k]].a;
      double chi2 = 0;
      cut_t r = px_eval(c, p, P, 3, c->layer[c->md.v[T->m[0]].module], &chi2, 0);
      if (r.pass && !(K3 && kept >= K3)) { px_t x = {p, o, chi2, r.margin}; VPUSH(c->pt3, x); ++kept; }
    }
  }
  return 0;
}

/* Indexed enumeration of the same (pLS, object) pairs: the definition above is all pairs; here a
 * pair is visited only if the object's FIRST anchor can pass its own residual cuts.  Per module the
 * bounding box of the event's MD anchors (rt, azimuth, z: measured from the MDs themselves, so no
 * premise about the geometry) is tested against the seed's extrapolation window with interval
 * arithmetic in fp64 and absolute margins (1e-6) far above rounding; objects are then visited in
 * the same order as the all-pairs loops (T3 / T5 are grouped by first MD, MDs by module), so the
 * result arrays are IDENTICAL, which tests/test_oracle_pins.py checks against lsto_link_pixel. */
typedef struct { double rlo, rhi, zlo, zhi, pref, dlo, dhi; int any; } mbox_t;

static int px_box_possible(const lsto_ctx *c, uint32_t p, const mbox_t *b, int cat) {
  const lsto_config *g = &c->cfg;
  const double M = 1e-6;
  double pt = c->spt[p], eta = c->seta[p], phi = c->sphi[p], z0 = c->sz0[p];
  if (!(pt > GUARD)) return 0;
  double kp = -(double)c->sq[p] * g->kB / (2.0 * pt), sh = sinh(eta);
  double s_lo, s_hi;          /* arc-length interval of an anchor inside the box */
  if (!is_endcap(cat)) {
    s_lo = arc_f(b->rlo, kp); s_hi = arc_f(b->rhi, kp);      /* increasing in rt */
  } else {
    if (!(fabs(sh) > GUARD)) return 0;
    double a = (b->zlo - z0) / sh, d = (b->zhi - z0) / sh;   /* linear in z */
    s_lo = min2(a, d); s_hi = max2(a, d);
  }
  if (!(s_hi > 0.0)) return 0;
  if (s_lo < 0.0) s_lo = 0.0;
  /* azimuth: predicted phi + kp s over [s_lo, s_hi] against the anchors' azimuth interval */
  double f_lo = phi + min2(kp * s_lo, kp * s_hi), f_hi = phi + max2(kp * s_lo, kp * s_hi);
  double sphi = g->seed_sig_phi + g->seed_sig_pt * fabs(kp) * s_hi + g->sig_t[cat] / b->rlo;
  double tol = g->n_sigma * sphi + M;
  double a_lo = b->pref + b->dlo, a_hi = b->pref + b->dhi;
  double width = (a_hi - a_lo) + (f_hi - f_lo) + 2.0 * tol;
  if (width < 2.0 * 3.14159265358979323846) {
    double mid = wrap_pi(0.5 * (a_lo + a_hi) - 0.5 * (f_lo + f_hi));
    if (fabs(mid) > 0.5 * width) return 0;
  }
  if (!is_endcap(cat)) {
    double z1 = z0 + sh * s_lo, z2 = z0 + sh * s_hi;
    double tz = g->n_sigma * (g->seed_sig_z + g->sig_z[cat]) + M;
    if (min2(z1, z2) - tz > b->zhi || max2(z1, z2) + tz < b->zlo) return 0;
  } else if (fabs(kp) * s_hi < 1.5) {          /* sin(kp s)/kp increases with s while |kp s| < pi/2 */
    double r1 = (fabs(kp * s_lo) <= 1e-4) ? s_lo : sin(kp * s_lo) / kp;
    double r2 = (fabs(kp * s_hi) <= 1e-4) ? s_hi : sin(kp * s_hi) / kp;
    double tr = g->n_sigma * (g->seed_sig_z / fabs(sh) + g->sig_r[cat]) + M;
    if (min2(r1, r2) - tr > b->rhi || max2(r1, r2) + tr < b->rlo) return 0;
  }
  return 1;
}

int lsto_link_pixel_indexed(lsto_ctx *c, uint32_t s0, uint32_t s1) {
  VCLEAR(c->pt5); VCLEAR(c->pt3);
  if (s1 > c->n_seeds) s1 = c->n_seeds;
  uint32_t nm = c->n_modules, nmd = c->md.n;
  mbox_t *box = calloc((size_t)nm + 1, sizeof(mbox_t));
  uint32_t *mods = malloc(((size_t)nm + 1) * 4), n_start = 0;
  for (uint32_t m = 0; m < nm; ++m) {
    if (!((c->cfg.start_layer_mask >> c->layer[m]) & 1u)) continue;
    uint32_t a = c->md_mod_off[m], b = c->md_mod_off[m + 1];
    if (a == b) continue;
    mbox_t *q = &box[m];
    const pt3 *f = &c->md.v[a].a;
    q->pref = atan2(f->y, f->x);
    q->rlo = q->rhi = f->rt; q->zlo = q->zhi = f->z; q->dlo = q->dhi = 0.0; q->any = 1;
    for (uint32_t i = a + 1; i < b; ++i) {
      const pt3 *h = &c->md.v[i].a;
      double d = wrap_pi(atan2(h->y, h->x) - q->pref);
      q->rlo = min2(q->rlo, h->rt); q->rhi = max2(q->rhi, h->rt);
      q->zlo = min2(q->zlo, h->z); q->zhi = max2(q->zhi, h->z);
      q->dlo = min2(q->dlo, d); q->dhi = max2(q->dhi, d);
    }
    mods[n_start++] = m;
  }
  /* T5 range of a first MD (T5 are built T3 by T3, so they ascend in their first MD) */
  uint32_t *t5_off = calloc((size_t)nmd + 2, 4);
  for (uint32_t i = 0; i < c->t5.n; ++i) t5_off[c->t5.v[i].m[0] + 1]++;
  for (uint32_t i = 0; i < nmd; ++i) t5_off[i + 1] += t5_off[i];
  for (int five = 1; five >= 0; --five) {
    for (uint32_t p = s0; p < s1; ++p) {
      const uint32_t K = c->trunc[five ? LSTO_PT5 : LSTO_PT3][0];       /* occupancy truncation: per pixel seed */
      uint32_t kept = 0;
      for (uint32_t k = 0; k < n_start; ++k) {
        uint32_t m = mods[k];
        if (!px_box_possible(c, p, &box[m], c->category[m])) continue;
        for (uint32_t i = c->md_mod_off[m]; i < c->md_mod_off[m + 1]; ++i) {
          uint32_t o0 = five ? t5_off[i] : c->t3_md_off[i], o1 = five ? t5_off[i + 1] : c->t3_md_off[i + 1];
          for (uint32_t o = o0; o < o1; ++o) {
            const pt3 *P[5];
            int n = five ? 5 : 3;
            const uint32_t *mm = five ? c->t5.v[o].m : c->t3.v[o].m;
            for (int q = 0; q < n; ++q) P[q] = &c->md.v[mm[q]].a;
            double chi2 = 0;
            cut_t r = px_eval(c, p, P, n, c->layer[m], &chi2, 0);
            if (r.pass && !(K && kept >= K)) { px_t x = {p, o, chi2, r.margin}; if (five) VPUSH(c->pt5, x); else VPUSH(c->pt3, x); ++kept; }
          }
        }
      }
    }
  }
  free(box); free(mods); free(t5_off);
  return 0;
}

/* ------------------------------------------------------------------ C7 duplicate removal, TC
 * cross-cleaning pT3 vs pT5; T5 vs pT5 + cleaned pT3; unused pLS vs all; close in
 * eta-phi, and objects must not share hits; TC = pT5 + pT3 + T5 + unlinked pLS. */
typedef struct {
  int n_ot, has_pls;
  uint32_t ot[10];
  uint32_t pix[4];
  uint32_t pls;
  double score, eta, phi;
} dobj_t;

static void t5_hits(const lsto_ctx *c, const t5_t *T, uint32_t *h) {
  for (int k = 0; k < 5; ++k) { h[2 * k] = c->md.v[T->m[k]].hl; h[2 * k + 1] = c->md.v[T->m[k]].hu; }
}
static void t3_hits(const lsto_ctx *c, const t3_t *T, uint32_t *h) {
  for (int k = 0; k < 3; ++k) { h[2 * k] = c->md.v[T->m[k]].hl; h[2 * k + 1] = c->md.v[T->m[k]].hu; }
}
static dobj_t dobj_t5(const lsto_ctx *c, uint32_t i) {
  dobj_t d; memset(&d, 0, sizeof(d));
  const t5_t *T = &c->t5.v[i];
  d.n_ot = 10; t5_hits(c, T, d.ot); d.score = T->chi2; d.eta = T->eta; d.phi = T->phi;
  return d;
}
static dobj_t dobj_px(const lsto_ctx *c, const px_t *x, int five) {
  dobj_t d; memset(&d, 0, sizeof(d));
  if (five) { d.n_ot = 10; t5_hits(c, &c->t5.v[x->obj], d.ot); }
  else { d.n_ot = 6; t3_hits(c, &c->t3.v[x->obj], d.ot); }
  d.has_pls = 1; d.pls = x->pls;
  for (int k = 0; k < 4; ++k) d.pix[k] = c->sids[4 * x->pls + k];
  d.score = x->chi2; d.eta = c->seta[x->pls]; d.phi = c->sphi[x->pls];
  return d;
}
static dobj_t dobj_pls(const lsto_ctx *c, uint32_t p) {
  dobj_t d; memset(&d, 0, sizeof(d));
  d.has_pls = 1; d.pls = p;
  for (int k = 0; k < 4; ++k) d.pix[k] = c->sids[4 * p + k];
  d.eta = c->seta[p]; d.phi = c->sphi[p];
  return d;
}
static int shared_ot(const dobj_t *a, const dobj_t *b) {
  int n = 0;
  for (int i = 0; i < a->n_ot; ++i) for (int j = 0; j < b->n_ot; ++j) if (a->ot[i] == b->ot[j]) ++n;
  return n;
}
static int shared_pix(const dobj_t *a, const dobj_t *b) {
  if (!a->has_pls || !b->has_pls) return 0;
  int n = 0;
  for (int i = 0; i < 4; ++i) {
    int hit = 0;
    for (int j = 0; j < 4; ++j) if (a->pix[i] == b->pix[j]) hit = 1;
    n += hit;
  }
  return n;
}
static double dr2_f(const dobj_t *a, const dobj_t *b) {
  double de = a->eta - b->eta, dp = wrap_pi(a->phi - b->phi);
  return de * de + dp * dp;
}
/* "b beats a": (score, key) lexicographic.  The scores use anchors only, so two objects that differ
 * in an upper hit tie exactly; the key must then not depend on the order in which the caller
 * listed the hits: key = OT hit coordinates (x, y, z of every hit in layer order), then - only for
 * objects identical in all coordinates - the pLS index and the hit indices (reading 15). */
static int beats(const lsto_ctx *c, const dobj_t *b, const dobj_t *a) {
  if (b->score < a->score) return 1;
  if (b->score > a->score) return 0;
  int n = a->n_ot < b->n_ot ? a->n_ot : b->n_ot;
  for (int k = 0; k < n; ++k) {
    uint32_t hb = b->ot[k], ha = a->ot[k];
    if (c->hx[hb] != c->hx[ha]) return c->hx[hb] < c->hx[ha];
    if (c->hy[hb] != c->hy[ha]) return c->hy[hb] < c->hy[ha];
    if (c->hz[hb] != c->hz[ha]) return c->hz[hb] < c->hz[ha];
  }
  if (a->has_pls && b->has_pls && b->pls != a->pls) return b->pls < a->pls;
  for (int k = 0; k < n; ++k) if (b->ot[k] != a->ot[k]) return b->ot[k] < a->ot[k];
  return 0;
}
/* cross-cleaning predicate: close in eta-phi OR sharing any hit */
static int cross_dup(const lsto_ctx *c, const dobj_t *a, const dobj_t *b, double *m) {
  double d = dr2_f(a, b);
  double rel = fabs(d - c->cfg.dr2max) / c->cfg.dr2max;
  if (rel < *m) *m = rel;
  return (d < c->cfg.dr2max) || shared_ot(a, b) >= 1 || shared_pix(a, b) >= 1;
}

/* S0 within one collection.  brute: all pairs.  indexed: pairs found through a hit -> objects
 * incidence list (plus same-pLS groups), which enumerates exactly the pairs sharing >= 1 OT hit. */
static void s0_clean(const lsto_ctx *c, const dobj_t *o, uint32_t n, int min_shared, int same_pls_rule,
                     int brute, uint8_t *keep) {
  for (uint32_t i = 0; i < n; ++i) keep[i] = 1;
  if (!c->cfg.s0_enabled || n == 0) return;
  if (brute) {
    for (uint32_t a = 0; a < n; ++a)
      for (uint32_t b = 0; b < n; ++b) {
        if (a == b) continue;
        int dup = (same_pls_rule && o[a].pls == o[b].pls) || shared_ot(&o[a], &o[b]) >= min_shared;
        if (dup && beats(c, &o[b], &o[a])) keep[a] = 0;
      }
    return;
  }
  /* incidence lists by OT hit */
  uint32_t nh = c->n_hits;
  uint32_t *off = calloc((size_t)nh + 2, 4);
  for (uint32_t a = 0; a < n; ++a) for (int k = 0; k < o[a].n_ot; ++k) off[o[a].ot[k] + 1]++;
  for (uint32_t h = 0; h < nh; ++h) off[h + 1] += off[h];
  uint32_t *lst = malloc(((size_t)off[nh] + 1) * 4), *fill = malloc(((size_t)nh + 1) * 4);
  memcpy(fill, off, ((size_t)nh + 1) * 4);
  for (uint32_t a = 0; a < n; ++a) for (int k = 0; k < o[a].n_ot; ++k) lst[fill[o[a].ot[k]]++] = a;
  for (uint32_t a = 0; a < n; ++a) {
    for (int k = 0; k < o[a].n_ot && keep[a]; ++k) {
      uint32_t h = o[a].ot[k];
      for (uint32_t e = off[h]; e < off[h + 1]; ++e) {
        uint32_t b = lst[e];
        if (b == a) continue;
        if (shared_ot(&o[a], &o[b]) >= min_shared && beats(c, &o[b], &o[a])) { keep[a] = 0; break; }
      }
    }
  }
  free(off); free(lst); free(fill);
  if (same_pls_rule) {
    /* objects of one pLS are contiguous (built seed by seed) */
    uint32_t a0 = 0;
    while (a0 < n) {
      uint32_t a1 = a0;
      while (a1 < n && o[a1].pls == o[a0].pls) ++a1;
      for (uint32_t a = a0; a < a1; ++a) for (uint32_t b = a0; b < a1; ++b)
        if (a != b && beats(c, &o[b], &o[a])) keep[a] = 0;
      a0 = a1;
    }
  }
}

/* S0, fix-point variant (SURVEY.md 8(f)3 "iterated dedup"; cleaning of PAPER.md:77-83).  The non-greedy
 * rule removes a when SOME better duplicate b exists, even a b that is itself removed by a still better c
 * that a does not overlap: a is lost for nothing.  The fix-point is the greedy definition: take the objects
 * from the best to the worst ("beats" is a strict total order); an object is kept iff no KEPT object is a
 * duplicate of it (shares >= min_shared OT hits).  Every kept object of the non-greedy rule is kept here
 * too.  Applied to the T5 collection (lsto_set_s0_fixpoint); the pixel-seeded collections keep the
 * non-greedy rule, whose same-seed clause already leaves one object per seed. */
static const lsto_ctx *g_sort_ctx;
static const dobj_t *g_sort_obj;
static int cmp_beats(const void *pa, const void *pb) {
  uint32_t a = *(const uint32_t *)pa, b = *(const uint32_t *)pb;
  if (a == b) return 0;
  return beats(g_sort_ctx, &g_sort_obj[a], &g_sort_obj[b]) ? -1 : 1;
}
static void s0_fixpoint(const lsto_ctx *c, const dobj_t *o, uint32_t n, int min_shared, uint8_t *keep) {
  for (uint32_t i = 0; i < n; ++i) keep[i] = 1;
  if (!c->cfg.s0_enabled || n == 0) return;
  uint32_t *order = malloc((size_t)n * 4), *rank = malloc((size_t)n * 4);
  for (uint32_t i = 0; i < n; ++i) order[i] = i;
  g_sort_ctx = c; g_sort_obj = o;
  qsort(order, n, 4, cmp_beats);
  for (uint32_t r = 0; r < n; ++r) rank[order[r]] = r;
  uint32_t nh = c->n_hits;
  uint32_t *off = calloc((size_t)nh + 2, 4);
  for (uint32_t a = 0; a < n; ++a) for (int k = 0; k < o[a].n_ot; ++k) off[o[a].ot[k] + 1]++;
  for (uint32_t h = 0; h < nh; ++h) off[h + 1] += off[h];
  uint32_t *lst = malloc(((size_t)off[nh] + 1) * 4), *fill = malloc(((size_t)nh + 1) * 4);
  memcpy(fill, off, ((size_t)nh + 1) * 4);
  for (uint32_t a = 0; a < n; ++a) for (int k = 0; k < o[a].n_ot; ++k) lst[fill[o[a].ot[k]]++] = a;
  for (uint32_t r = 0; r < n; ++r) {                     /* best first: every better object is already decided */
    uint32_t a = order[r];
    for (int k = 0; k < o[a].n_ot && keep[a]; ++k) {
      uint32_t h = o[a].ot[k];
      for (uint32_t e = off[h]; e < off[h + 1]; ++e) {
        uint32_t b = lst[e];
        if (b != a && rank[b] < r && keep[b] && shared_ot(&o[a], &o[b]) >= min_shared) { keep[a] = 0; break; }
      }
    }
  }
  free(order); free(rank); free(off); free(lst); free(fill);
}
int lsto_set_s0_fixpoint(lsto_ctx *c, int on) { if (!c) return -1; c->s0_fixpoint = on != 0; return 0; }

int lsto_dedup(lsto_ctx *c, int brute) {
  uint32_t n5 = c->t5.n, np5 = c->pt5.n, np3 = c->pt3.n, ns = c->n_seeds;
  free(c->keep_t5); free(c->keep_pt3); free(c->keep_pt5); free(c->keep_pls);
  c->keep_t5 = malloc((size_t)n5 + 1); c->keep_pt5 = malloc((size_t)np5 + 1);
  c->keep_pt3 = malloc((size_t)np3 + 1); c->keep_pls = malloc((size_t)ns + 1);
  dobj_t *o5 = malloc(((size_t)n5 + 1) * sizeof(dobj_t)), *op5 = malloc(((size_t)np5 + 1) * sizeof(dobj_t));
  dobj_t *op3 = malloc(((size_t)np3 + 1) * sizeof(dobj_t));
  for (uint32_t i = 0; i < n5; ++i) o5[i] = dobj_t5(c, i);
  for (uint32_t i = 0; i < np5; ++i) op5[i] = dobj_px(c, &c->pt5.v[i], 1);
  for (uint32_t i = 0; i < np3; ++i) op3[i] = dobj_px(c, &c->pt3.v[i], 0);
  double m = INFINITY;
  /* S0 intra-collection */
  if (c->s0_fixpoint && !brute) s0_fixpoint(c, o5, n5, c->cfg.dup_t5_shared, c->keep_t5);
  else s0_clean(c, o5, n5, c->cfg.dup_t5_shared, 0, brute, c->keep_t5);
  s0_clean(c, op5, np5, c->cfg.dup_pt5_shared, 1, brute, c->keep_pt5);
  s0_clean(c, op3, np3, c->cfg.dup_pt3_shared, 1, brute, c->keep_pt3);
  /* S1: pT3 vs pT5 (both S0 survivors) */
  uint8_t *k3 = malloc((size_t)np3 + 1);
  memcpy(k3, c->keep_pt3, np3);
  for (uint32_t a = 0; a < np3; ++a) {
    if (!c->keep_pt3[a]) continue;
    for (uint32_t b = 0; b < np5; ++b)
      if (c->keep_pt5[b] && cross_dup(c, &op3[a], &op5[b], &m)) { k3[a] = 0; break; }
  }
  memcpy(c->keep_pt3, k3, np3);
  free(k3);
  /* S2: T5 vs pT5 survivors and pT3 survivors of S1 */
  uint8_t *k5 = malloc((size_t)n5 + 1);
  memcpy(k5, c->keep_t5, n5);
  for (uint32_t a = 0; a < n5; ++a) {
    if (!c->keep_t5[a]) continue;
    int dup = 0;
    for (uint32_t b = 0; b < np5 && !dup; ++b) if (c->keep_pt5[b] && cross_dup(c, &o5[a], &op5[b], &m)) dup = 1;
    for (uint32_t b = 0; b < np3 && !dup; ++b) if (c->keep_pt3[b] && cross_dup(c, &o5[a], &op3[b], &m)) dup = 1;
    if (dup) k5[a] = 0;
  }
  memcpy(c->keep_t5, k5, n5);
  free(k5);
  /* S3: unused pLS (constituent of no created pT3 / pT5) vs survivors, and vs earlier unused pLS */
  uint8_t *used = calloc((size_t)ns + 1, 1);
  for (uint32_t i = 0; i < np5; ++i) used[c->pt5.v[i].pls] = 1;
  for (uint32_t i = 0; i < np3; ++i) used[c->pt3.v[i].pls] = 1;
  for (uint32_t a = 0; a < ns; ++a) {
    c->keep_pls[a] = 0;
    if (used[a]) continue;
    dobj_t A = dobj_pls(c, a);
    int dup = 0;
    for (uint32_t b = 0; b < np5 && !dup; ++b) if (c->keep_pt5[b] && cross_dup(c, &A, &op5[b], &m)) dup = 1;
    for (uint32_t b = 0; b < np3 && !dup; ++b) if (c->keep_pt3[b] && cross_dup(c, &A, &op3[b], &m)) dup = 1;
    for (uint32_t b = 0; b < n5 && !dup; ++b) if (c->keep_t5[b] && cross_dup(c, &A, &o5[b], &m)) dup = 1;
    for (uint32_t b = 0; b < a && !dup; ++b) {
      if (used[b]) continue;
      dobj_t Bq = dobj_pls(c, b);
      if (dr2_f(&A, &Bq) < c->cfg.dr2max) dup = 1;
    }
    c->keep_pls[a] = !dup;
  }
  free(used);
  /* S4: TC = pT5, pT3, T5, pLS survivors */
  VCLEAR(c->tc);
  for (uint32_t i = 0; i < np5; ++i) if (c->keep_pt5[i]) {
    uint32_t p = c->pt5.v[i].pls; tc_t t = {LSTO_PT5, i, c->spt[p], c->seta[p], c->sphi[p]}; VPUSH(c->tc, t); }
  for (uint32_t i = 0; i < np3; ++i) if (c->keep_pt3[i]) {
    uint32_t p = c->pt3.v[i].pls; tc_t t = {LSTO_PT3, i, c->spt[p], c->seta[p], c->sphi[p]}; VPUSH(c->tc, t); }
  for (uint32_t i = 0; i < n5; ++i) if (c->keep_t5[i]) {
    const t5_t *T = &c->t5.v[i]; tc_t t = {LSTO_T5, i, T->pt, T->eta, T->phi}; VPUSH(c->tc, t); }
  for (uint32_t p = 0; p < ns; ++p) if (c->keep_pls[p]) {
    tc_t t = {LSTO_TC, p, c->spt[p], c->seta[p], c->sphi[p]}; VPUSH(c->tc, t); }
  free(o5); free(op5); free(op3);
  return 0;
}

/* ------------------------------------------------------------------ getters */
uint32_t lsto_arity(int level) {
  switch (level) {
    case LSTO_MD: return 2; case LSTO_LS: return 4; case LSTO_T3: return 6; case LSTO_T5: return 10;
    case LSTO_PT3: return 6; case LSTO_PT5: return 10; default: return 0;
  }
}
uint32_t lsto_count(const lsto_ctx *c, int level) {
  switch (level) {
    case LSTO_MD: return c->md.n; case LSTO_LS: return c->ls.n; case LSTO_T3: return c->t3.n;
    case LSTO_T5: return c->t5.n; case LSTO_PT3: return c->pt3.n; case LSTO_PT5: return c->pt5.n;
    case LSTO_TC: return c->tc.n; default: return 0;
  }
}
static void md_hits(const lsto_ctx *c, uint32_t m, uint32_t *h) { h[0] = c->md.v[m].hl; h[1] = c->md.v[m].hu; }

int lsto_get(const lsto_ctx *c, int level, uint32_t *hit_idx, uint32_t *parents, double *f, double *margin) {
  uint32_t n = lsto_count(c, level);
  for (uint32_t i = 0; i < n; ++i) {
    double ff[4] = {0, 0, 0, 0}, mg = 0;
    uint32_t par[2] = {0, 0};
    uint32_t h[10];
    switch (level) {
      case LSTO_MD: { const md_t *o = &c->md.v[i]; h[0] = o->hl; h[1] = o->hu; par[0] = o->module;
        ff[0] = o->dphi; ff[1] = o->kappa; ff[2] = o->sigk; mg = o->margin; break; }
      case LSTO_LS: { const ls_t *o = &c->ls.v[i]; md_hits(c, o->mi, h); md_hits(c, o->mo, h + 2);
        par[0] = o->mi; par[1] = o->mo; ff[0] = o->dphi; ff[1] = o->kappa; ff[2] = o->sigk; mg = o->margin; break; }
      case LSTO_T3: { const t3_t *o = &c->t3.v[i]; t3_hits(c, o, h); par[0] = o->la; par[1] = o->lb;
        ff[0] = o->beta; ff[1] = o->kappa3; ff[2] = o->sigk3; mg = o->margin; break; }
      case LSTO_T5: { const t5_t *o = &c->t5.v[i]; t5_hits(c, o, h); par[0] = o->ta; par[1] = o->tb;
        ff[0] = o->R; ff[1] = o->chi2; ff[2] = o->k3a; ff[3] = o->k3b; mg = o->margin; break; }
      case LSTO_PT3: { const px_t *o = &c->pt3.v[i]; t3_hits(c, &c->t3.v[o->obj], h); par[0] = o->pls; par[1] = o->obj;
        ff[0] = o->chi2; mg = o->margin; break; }
      case LSTO_PT5: { const px_t *o = &c->pt5.v[i]; t5_hits(c, &c->t5.v[o->obj], h); par[0] = o->pls; par[1] = o->obj;
        ff[0] = o->chi2; mg = o->margin; break; }
      case LSTO_TC: { const tc_t *o = &c->tc.v[i]; par[0] = o->type; par[1] = o->obj;
        ff[0] = o->pt; ff[1] = o->eta; ff[2] = o->phi; ff[3] = (double)o->type; break; }
      default: return -1;
    }
    uint32_t ar = lsto_arity(level);
    if (hit_idx) for (uint32_t k = 0; k < ar; ++k) hit_idx[(size_t)i * ar + k] = h[k];
    if (parents) { parents[2 * (size_t)i] = par[0]; parents[2 * (size_t)i + 1] = par[1]; }
    if (f) for (int k = 0; k < 4; ++k) f[4 * (size_t)i + k] = ff[k];
    if (margin) margin[i] = mg;
  }
  return 0;
}
int lsto_get_t5_kin(const lsto_ctx *c, double *out) {
  for (uint32_t i = 0; i < c->t5.n; ++i) {
    out[3 * (size_t)i] = c->t5.v[i].pt; out[3 * (size_t)i + 1] = c->t5.v[i].eta; out[3 * (size_t)i + 2] = c->t5.v[i].phi;
  }
  return 0;
}
int lsto_get_keep(const lsto_ctx *c, int level, uint8_t *keep) {
  const uint8_t *src; uint32_t n;
  switch (level) {
    case LSTO_T5: src = c->keep_t5; n = c->t5.n; break;
    case LSTO_PT3: src = c->keep_pt3; n = c->pt3.n; break;
    case LSTO_PT5: src = c->keep_pt5; n = c->pt5.n; break;
    case -1: src = c->keep_pls; n = c->n_seeds; break;
    default: return -1;
  }
  if (!src) return -2;
  memcpy(keep, src, n);
  return 0;
}

/* ------------------------------------------------------------------ single-candidate evaluation */
static void merge(cut_t *r, cut_t s) { if (!s.pass) r->pass = 0; if (s.margin < r->margin) r->margin = s.margin; }

int lsto_eval(const lsto_ctx *c, int level, const uint32_t *hits, uint32_t seed, double *margin) {
  int nmd;
  switch (level) {
    case LSTO_MD: nmd = 1; break; case LSTO_LS: nmd = 2; break;
    case LSTO_T3: case LSTO_PT3: nmd = 3; break; case LSTO_T5: case LSTO_PT5: nmd = 5; break;
    default: return -1;
  }
  cut_t r = {1, INFINITY};
  md_t md[5];
  for (int k = 0; k < nmd; ++k) {
    uint32_t hl = hits[2 * k], hu = hits[2 * k + 1];
    if (hl >= c->n_hits || hu >= c->n_hits) return -1;
    uint32_t dl = c->hdet[hl], du = c->hdet[hu];
    memset(&md[k], 0, sizeof(md_t));
    if ((dl & 1u) != 0 || du != dl + 1) { r.pass = 0; continue; }
    uint32_t m = dl >> 1;
    int cat = c->category[m];
    pt3 l = hit_pt(c, hl, cat), u = hit_pt(c, hu, cat);
    md[k].hl = hl; md[k].hu = hu; md[k].module = m;
    merge(&r, md_eval(c, &l, &u, cat, &md[k]));
  }
  if (!r.pass && r.margin == INFINITY) { if (margin) *margin = r.margin; return 0; }
  ls_t ls[4];
  for (int k = 0; k + 1 < nmd; ++k) {
    if (!map_has(c, md[k].module, md[k + 1].module)) r.pass = 0;
    memset(&ls[k], 0, sizeof(ls_t));
    merge(&r, ls_eval(c, &md[k], &md[k + 1], &ls[k]));
  }
  t3_t t3[3];
  for (int k = 0; k + 2 < nmd; k += 2) {
    memset(&t3[k / 2], 0, sizeof(t3_t));
    merge(&r, t3_eval(c, &md[k].a, &md[k + 1].a, &md[k + 2].a, &t3[k / 2]));
  }
  const pt3 *P[5];
  for (int k = 0; k < nmd; ++k) P[k] = &md[k].a;
  if (nmd == 5) {
    t5_t t5; memset(&t5, 0, sizeof(t5));
    merge(&r, t5_eval(c, P, t3[0].kappa3, t3[0].sigk3, t3[1].kappa3, t3[1].sigk3, &t5));
  }
  if (level == LSTO_PT3 || level == LSTO_PT5) {
    if (seed >= c->n_seeds) return -1;
    double chi2 = 0;
    merge(&r, px_eval(c, seed, P, nmd, c->layer[md[0].module], &chi2, 1));
  }
  if (margin) *margin = r.margin;
  return r.pass;
}

/* ------------------------------------------------------------------ test hooks (pins only)
 * Expose the C0 helpers and the Kasa fit on double inputs so that tests can pin them to closed
 * forms without going through fp32 hit rounding. */
void lsto_test_helpers(const double *A, const double *B, const double *Cc, double k, double *out) {
  pt3 a = {A[0], A[1], A[2], hypot(A[0], A[1]), 0}, b = {B[0], B[1], B[2], hypot(B[0], B[1]), 0};
  pt3 cc = {Cc[0], Cc[1], Cc[2], hypot(Cc[0], Cc[1]), 0};
  out[0] = sd_f(&a, &b);
  out[1] = dphi_f(&a, &b);
  out[2] = chord_f(&a, &b);
  out[3] = dr_f(&a, &b);
  out[4] = kappa3_f(&a, &b, &cc);
  out[5] = arc_f(a.rt, k);
  out[6] = wrap_pi(k);
}
int lsto_test_kasa(const lsto_config *cfg, const double *x, const double *y, const int32_t *cat, double kc,
                   double *R, double *chi2) {
  lsto_ctx c; memset(&c, 0, sizeof(c));
  c.cfg = *cfg;
  c.kmax = cfg->kB / (2.0 * cfg->pt_min);
  pt3 p[5]; const pt3 *P[5];
  for (int k = 0; k < 5; ++k) { p[k].x = x[k]; p[k].y = y[k]; p[k].z = 0; p[k].rt = hypot(x[k], y[k]); p[k].cat = cat[k]; P[k] = &p[k]; }
  double detn = 0;
  return kasa_fit(&c, P, kc, R, chi2, &detn);
}

/* Evaluate ONE selection function on double inputs (no event, no fp32 rounding) and return every cut
 * it evaluated as (kind, v, thr) triples in evaluation order (see trace_push).  level: LSTO_MD
 * (pts = lower, upper; cats[0] = module category), LSTO_LS (pts = anchors i, o; aux = kappa_MD(i),
 * sigma(i), kappa_MD(o), sigma(o)), LSTO_T3 (3 anchors), LSTO_T5 (5 anchors; aux = kappa3(a),
 * sigma(a), kappa3(b), sigma(b)), LSTO_PT3 / LSTO_PT5 (3 / 5 anchors; aux = pt, eta, phi, z0, q,
 * logical layer of the first MD).  out_f (8 doubles): MD / LS {dphi, kappa, sigk}; T3 {beta, kappa3,
 * sigk3}; T5 {R, chi2, pt, eta, phi}; PT3 / PT5 {chi2_pix}.  Returns pass (0 / 1), -1 on bad level. */
int lsto_test_cuts(const lsto_config *cfg, int level, const double *pts, const int32_t *cats, const double *aux,
                   double *out_f, double *trace, int trace_cap, int *n_trace) {
  lsto_ctx c; memset(&c, 0, sizeof(c));
  c.cfg = *cfg;
  c.kmax = cfg->kB / (2.0 * cfg->pt_min);
  int npts = level == LSTO_MD || level == LSTO_LS ? 2 : (level == LSTO_T3 || level == LSTO_PT3 ? 3 :
             (level == LSTO_T5 || level == LSTO_PT5 ? 5 : 0));
  if (!npts) return -1;
  pt3 p[5]; const pt3 *P[5];
  for (int k = 0; k < npts; ++k) {
    p[k].x = pts[3 * k]; p[k].y = pts[3 * k + 1]; p[k].z = pts[3 * k + 2];
    p[k].rt = sqrt(p[k].x * p[k].x + p[k].y * p[k].y);
    p[k].cat = cats[level == LSTO_MD ? 0 : k];
    P[k] = &p[k];
  }
  for (int k = 0; k < 8; ++k) out_f[k] = 0.0;
  g_trace = trace; g_trace_n = 0; g_trace_cap = trace_cap;
  cut_t r;
  if (level == LSTO_MD) {
    md_t o; memset(&o, 0, sizeof(o));
    r = md_eval(&c, &p[0], &p[1], cats[0], &o);
    out_f[0] = o.dphi; out_f[1] = o.kappa; out_f[2] = o.sigk;
  } else if (level == LSTO_LS) {
    md_t mi, mo; memset(&mi, 0, sizeof(mi)); memset(&mo, 0, sizeof(mo));
    mi.a = p[0]; mi.kappa = aux[0]; mi.sigk = aux[1];
    mo.a = p[1]; mo.kappa = aux[2]; mo.sigk = aux[3];
    ls_t o; memset(&o, 0, sizeof(o));
    r = ls_eval(&c, &mi, &mo, &o);
    out_f[0] = o.dphi; out_f[1] = o.kappa; out_f[2] = o.sigk;
  } else if (level == LSTO_T3) {
    t3_t o; memset(&o, 0, sizeof(o));
    r = t3_eval(&c, P[0], P[1], P[2], &o);
    out_f[0] = o.beta; out_f[1] = o.kappa3; out_f[2] = o.sigk3;
  } else if (level == LSTO_T5) {
    t5_t o; memset(&o, 0, sizeof(o));
    r = t5_eval(&c, P, aux[0], aux[1], aux[2], aux[3], &o);
    out_f[0] = o.R; out_f[1] = o.chi2; out_f[2] = o.pt; out_f[3] = o.eta; out_f[4] = o.phi;
  } else {
    double spt = aux[0], seta = aux[1], sphi = aux[2], sz0 = aux[3];
    int8_t sq = (int8_t)aux[4];
    c.spt = &spt; c.seta = &seta; c.sphi = &sphi; c.sz0 = &sz0; c.sq = &sq; c.n_seeds = 1;
    double chi2 = 0.0;
    r = px_eval(&c, 0, P, npts, (int)aux[5], &chi2, 1);
    out_f[0] = chi2;
  }
  if (n_trace) *n_trace = g_trace_n / 3;
  g_trace = NULL; g_trace_n = 0; g_trace_cap = 0;
  return r.pass;
}

/* Replace the object collections of the loaded event by hand-built ones, so that lsto_dedup can be
 * pinned on constructed cases (shared-hit thresholds, Delta R^2 edge, the pLS rules).  MDs are given
 * by their hit indices; T3 / T5 by MD indices (+ chi2, pt, eta, phi for T5); pT3 / pT5 by (pLS,
 * object index, chi2_pix), grouped by pLS as lsto_link_pixel builds them. */
int lsto_test_inject(lsto_ctx *c, uint32_t n_md, const uint32_t *md_hits, uint32_t n_t3, const uint32_t *t3_md,
                     uint32_t n_t5, const uint32_t *t5_md, const double *t5_kin /* chi2, pt, eta, phi */,
                     uint32_t n_pt3, const uint32_t *pt3_po, const double *pt3_chi2,
                     uint32_t n_pt5, const uint32_t *pt5_po, const double *pt5_chi2) {
  VCLEAR(c->md); VCLEAR(c->ls); VCLEAR(c->t3); VCLEAR(c->t5); VCLEAR(c->pt3); VCLEAR(c->pt5); VCLEAR(c->tc);
  for (uint32_t i = 0; i < n_md; ++i) {
    md_t m; memset(&m, 0, sizeof(m));
    m.hl = md_hits[2 * i]; m.hu = md_hits[2 * i + 1];
    if (m.hl >= c->n_hits || m.hu >= c->n_hits) return -1;
    m.module = c->hdet[m.hl] >> 1;
    m.a = hit_pt(c, m.hl, c->category[m.module]);
    VPUSH(c->md, m);
  }
  for (uint32_t i = 0; i < n_t3; ++i) {
    t3_t t; memset(&t, 0, sizeof(t));
    for (int k = 0; k < 3; ++k) { t.m[k] = t3_md[3 * i + k]; if (t.m[k] >= n_md) return -1; }
    VPUSH(c->t3, t);
  }
  for (uint32_t i = 0; i < n_t5; ++i) {
    t5_t t; memset(&t, 0, sizeof(t));
    for (int k = 0; k < 5; ++k) { t.m[k] = t5_md[5 * i + k]; if (t.m[k] >= n_md) return -1; }
    t.chi2 = t5_kin[4 * i]; t.pt = t5_kin[4 * i + 1]; t.eta = t5_kin[4 * i + 2]; t.phi = t5_kin[4 * i + 3];
    VPUSH(c->t5, t);
  }
  for (uint32_t i = 0; i < n_pt3; ++i) {
    px_t x = {pt3_po[2 * i], pt3_po[2 * i + 1], pt3_chi2[i], 0.0};
    if (x.pls >= c->n_seeds || x.obj >= n_t3) return -1;
    VPUSH(c->pt3, x);
  }
  for (uint32_t i = 0; i < n_pt5; ++i) {
    px_t x = {pt5_po[2 * i], pt5_po[2 * i + 1], pt5_chi2[i], 0.0};
    if (x.pls >= c->n_seeds || x.obj >= n_t5) return -1;
    VPUSH(c->pt5, x);
  }
  return 0;
}
