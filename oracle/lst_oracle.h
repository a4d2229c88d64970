/* lst_oracle.h -- CPU oracle for the Segment Linking / Line Segment Tracking hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded C, fp64 on the fp32 inputs
 * (every input is promoted to double before the first subtraction).  It follows
 * arxiv 2209.13711 section 2.1 step by step, with every formula and constant
 * the paper leaves open taken from the readings listed in DESIGN.md ("Readings of the
 * paper", = SURVEY.md 8(c) C0-C7).  It shares no code, header, table or constant
 * generator with the CUDA path under paper_2209_13711_b200/ and neither imports the
 * other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call it.
 *
 * Parity pins, function by function (DESIGN.md section 3 has the table):
 *   tests/test_oracle_pins.py        helix closed forms, noiseless-track chains, pT edge of B2 on
 *                                    generated hits, brute-force enumeration, permutation
 *                                    invariance, Kasa fit vs an independent geometric fit
 *   tests/test_oracle_pins2.py       two-sided pins: closed-form EDGE of B2, E2, L2 (mode R and Z),
 *                                    T3-1, T5-1, chi2max; every tolerance term of B1, E1, L1, L2, L3,
 *                                    sigma_kappa3, E_phi, E_z, sigma_phi_k, sigma_zeta_k ONE AT A TIME
 *                                    (the constants are data); closed forms of dphi_MD, beta, mode-Z
 *                                    kappa_LS, endcap kappa_MD; S0-S3 on hand-built collections;
 *                                    truth efficiency >= 99 % at every level on smeared events
 *   tests/test_oracle_restatement.py every cut variable and threshold against a third transcription
 *                                    of SURVEY.md 8(c) in numpy, on 1e4 candidates per level
 *   tests/test_oracle_mutations.py   30 single-token mutants of this file are each caught by the pin
 *                                    named for the mutated function
 * "parity unpinned" against the paper's own VALUES: the paper prints no cut value, object count
 * or worked example on data available here.
 */
#ifndef LST_ORACLE_H
#define LST_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  double kB;            /* 0.00299792458 * 3.8 GeV/cm                       (C0) */
  double pt_min;        /* 0.8 GeV                                  */
  double n_sigma;       /* 4                                                     */
  double z0max;         /* 15 cm                                                 */
  double d0max;         /* 2.5 cm                                                */
  double chi2max;       /* 18.42                                                 */
  double dr2max;        /* 1e-4                                                  */
  double map_kscale;    /* 1.25   (C2)                                           */
  double map_z0;        /* 20 cm  (C2)                                           */
  double ec_md_sys;     /* 0.3    (C3 L3)                                        */
  double modez_slack;   /* 0.15   (C3 L3)                                        */
  double seed_sig_phi;  /* 0.001  (C6)                                           */
  double seed_sig_pt;   /* 0.01   (C6)                                           */
  double seed_sig_z;    /* 0.05   (C6)                                           */
  double sig_t[4];      /* per category bPS,b2S,ePS,e2S: {.01,.009,.01,.009}/sqrt12 */
  double sig_z[4];      /* {.15, 5, 0, 0}/sqrt12                                 */
  double sig_r[4];      /* {0, 0, .15, 5}/sqrt12                                 */
  int32_t dup_t5_shared;   /* 5 */
  int32_t dup_pt5_shared;  /* 5 */
  int32_t dup_pt3_shared;  /* 3 */
  int32_t s0_enabled;      /* 1 */
  uint32_t start_layer_mask; /* bit L set: logical layer L may start a pT3/pT5 (C6) */
} lsto_config;

typedef struct lsto_ctx lsto_ctx;

enum { LSTO_MD = 0, LSTO_LS, LSTO_T3, LSTO_T5, LSTO_PT3, LSTO_PT5, LSTO_TC, LSTO_NLEVEL };

void lsto_default_config(lsto_config *c);

/* C2: module map from module boxes.  Returns CSR in malloc'd arrays (free with lsto_free). */
int lsto_build_module_map(uint32_t n_modules, const uint8_t *category, const uint8_t *layer,
                          const float *rmin, const float *rmax, const float *phic,
                          const float *half_phi, const float *zmin, const float *zmax,
                          const lsto_config *cfg, uint32_t **row_offsets, uint32_t **cols);
void lsto_free(void *p);

lsto_ctx *lsto_create(uint32_t n_modules, const uint8_t *category, const uint8_t *layer,
                      const uint32_t *map_offsets, const uint32_t *map_cols,
                      const lsto_config *cfg);
void lsto_destroy(lsto_ctx *c);

/* PAPER.md:125 occupancy truncation (optional; see the .c file): hit order inside a sensor = ascending
 * azimuth relative to phic[module]; caps[level * 16 + logical layer] = K keeps the first K objects of a
 * module (pixel levels: caps[level * 16] per seed); NULL caps = order only.  Call before lsto_load_event. */
int lsto_set_truncation(lsto_ctx *c, const float *phic, const uint32_t *caps);

int lsto_load_event(lsto_ctx *c, uint32_t n_hits, const float *x, const float *y, const float *z,
                    const uint32_t *det, uint32_t n_seeds, const float *pt, const float *eta,
                    const float *phi, const float *z0, const int8_t *q, const uint32_t *hit_ids);

/* stages; brute = 1 uses the all-pairs definition instead of the index-driven enumeration */
int lsto_build_md(lsto_ctx *c);
int lsto_build_ls(lsto_ctx *c, int brute);
int lsto_build_t3(lsto_ctx *c, int brute);
int lsto_build_t5(lsto_ctx *c, int brute);
int lsto_link_pixel(lsto_ctx *c, uint32_t seed_begin, uint32_t seed_end); /* pT5 then pT3: ALL pairs */
/* the same pairs through a per-module first-anchor window (identical output; see the .c file) */
int lsto_link_pixel_indexed(lsto_ctx *c, uint32_t seed_begin, uint32_t seed_end);
int lsto_dedup(lsto_ctx *c, int brute);                                   /* S0-S4 -> TC    */
/* S0 of the T5 collection as a fix-point (greedy from the best object down: kept iff no KEPT object is a
 * duplicate) instead of the non-greedy rule; see the .c file.  Ignored by the brute mode. */
int lsto_set_s0_fixpoint(lsto_ctx *c, int on);

uint32_t lsto_count(const lsto_ctx *c, int level);
/* copy-out: any pointer may be NULL.  hit_idx: n*arity original hit indices in layer order
 * (MD 2, LS 4, T3 6, T5 10, PT3 6 OT hits, PT5 10 OT hits); parents: MD {module}, LS {md_i,md_o},
 * T3 {ls_a,ls_b}, T5 {t3_a,t3_b}, PT3/PT5 {pls,obj}, TC {type,obj}; f: n*4 doubles:
 * MD {dphi,kappa,sigk,0} LS {dphi,kappa,sigk,0} T3 {beta,kappa3,sigk3,0} T5 {R,chi2,k3a,k3b}
 * PT3/PT5 {chi2pix,0,0,0} TC {pt,eta,phi,type}; margin: n doubles (min relative distance of any
 * cut variable to its threshold). */
int lsto_get(const lsto_ctx *c, int level, uint32_t *hit_idx, uint32_t *parents, double *f,
             double *margin);
uint32_t lsto_arity(int level);
/* T5 kinematics used by the cleaning (pt, eta, phi) */
int lsto_get_t5_kin(const lsto_ctx *c, double *pt_eta_phi /* n*3 */);
/* keep flags after S0..S3 for T5, PT3, PT5 and for pLS (level = -1, n_seeds entries) */
int lsto_get_keep(const lsto_ctx *c, int level, uint8_t *keep);

/* single-candidate evaluation on original hit indices; returns pass (1/0), fills margin.
 * MD: 2 hits; LS: 4; T3: 6; T5: 10; PT3: seed + 6; PT5: seed + 10.  Constituent objects are
 * evaluated too (a T3 passes only if both its LS and its 3 MDs pass). */
int lsto_eval(const lsto_ctx *c, int level, const uint32_t *hits, uint32_t seed, double *margin);

/* test hooks: C0 helpers {sd, dphi, chord, dr, kappa3, arc(rt_A;k), wrap(k)} and the Kasa fit */
void lsto_test_helpers(const double *A, const double *B, const double *C, double k, double *out7);
int lsto_test_kasa(const lsto_config *cfg, const double *x, const double *y, const int32_t *cat, double kc,
                   double *R, double *chi2);

/* test hooks (pins only): one selection function on double inputs with the trace of its cuts, and
 * hand-built object collections for lsto_dedup; see the .c file */
int lsto_test_cuts(const lsto_config *cfg, int level, const double *pts, const int32_t *cats, const double *aux,
                   double *out_f, double *trace, int trace_cap, int *n_trace);
int lsto_test_inject(lsto_ctx *c, uint32_t n_md, const uint32_t *md_hits, uint32_t n_t3, const uint32_t *t3_md,
                     uint32_t n_t5, const uint32_t *t5_md, const double *t5_kin,
                     uint32_t n_pt3, const uint32_t *pt3_po, const double *pt3_chi2,
                     uint32_t n_pt5, const uint32_t *pt5_po, const double *pt5_chi2);

/* TC entry types (parents[0] of level LSTO_TC) */
enum { LSTO_TC_T5 = LSTO_T5, LSTO_TC_PT3 = LSTO_PT3, LSTO_TC_PT5 = LSTO_PT5, LSTO_TC_PLS = LSTO_TC };

#ifdef __cplusplus
}
#endif
#endif
