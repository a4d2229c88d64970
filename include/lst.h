/* lst.h -- C-ABI of the B200-native Segment Linking / Line Segment Tracking hot path.
 *
 * Method: arxiv 2209.13711 section 2.1: mini-doublets (MD) ->
 * line segments (LS, :53-55,71) -> triplets (T3, :73) -> quintuplets (T5, :73) -> pixel-seeded
 * pT5 / pT3 (:75) -> duplicate removal and track candidates (TC, :77-83).  Every formula and
 * constant the paper leaves open is a reading listed in DESIGN.md ("Readings", C0-C7).
 *
 * Conventions
 *   - plain C, no torch types.  Every pointer argument says whether it is HOST or DEVICE memory.
 *   - every call returns LST_OK (0) or a negative lst_status; nothing throws or aborts; out-params
 *     are untouched on error.  lst_strerror() gives text (for LST_ECUDA: the CUDA error string).
 *   - units: cm, GeV, Tesla, radians.  Hits are fp32; indices are uint32.
 *   - one context = one detector (+ module map) on the CUDA device current at lst_create();
 *     a context owns n_slots independent event slots; calls on different slots may be issued
 *     on different CUDA streams concurrently ("multi-streaming").  Calls on
 *     one slot must be issued in order load -> run -> get from one host thread at a time;
 *     different slots may be driven from different host threads (nothing shared is written after
 *     lst_bind_workspace, which captures the slot's CUDA graph; concurrent lst_bind_workspace calls
 *     on one context are serialised inside the library).
 *   - the library never allocates device memory after lst_create(): each slot works inside one
 *     caller-provided workspace (lst_workspace_bytes / lst_bind_workspace).
 */
#ifndef LST_H
#define LST_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  LST_OK = 0,
  LST_EINVAL = -1,  /* null pointer, out-of-range index, unsorted map, bad geometry; per event: det >=
                       2*n_modules, NaN / infinite input, lower-sensor hit outside its module's box  */
  LST_ENOMEM = -2,  /* workspace too small, or an object collection overflowed its capacity     */
  LST_ECUDA = -3,   /* a CUDA call failed (sticky; text via lst_strerror)                       */
  LST_ESTATE = -4   /* call order violated (run before load, get before run, unbound workspace) */
} lst_status;

/* object levels */
typedef enum { LST_MD = 0, LST_LS, LST_T3, LST_T5, LST_PT3, LST_PT5, LST_TC, LST_NLEVEL } lst_level;

/* Selection constants (DESIGN.md Readings C0-C7).  lst_default_config fills
 * the defaults; per-category arrays are indexed by module category 0 bPS, 1 b2S, 2 ePS, 3 e2S. */
typedef struct {
  double kB;            /* 0.00299792458 * B[T] GeV/cm (B = 3.8 T)                                */
  double pt_min;        /* 0.8 GeV: the stub window of PAPER.md:37                                */
  double n_sigma;       /* 4: number of sigmas in every tolerance                                 */
  double z0max;         /* 15 cm: luminous-region half length used by MD / LS pointing cuts       */
  double d0max;         /* 2.5 cm: displacement allowance (module map, T3-2)                      */
  double chi2max;       /* 18.42: T5 circle-fit chi2 cut                                          */
  double dr2max;        /* 1e-4: "close in eta-phi" of PAPER.md:77, as Delta R^2                  */
  double map_kscale;    /* 1.25: curvature margin of the module map                               */
  double map_z0;        /* 20 cm: z0 margin of the module map                                     */
  double ec_md_sys;     /* 0.3: endcap-MD curvature systematic in LS cut L3                       */
  double modez_slack;   /* 0.15: mode-Z slack in LS cut L3                                        */
  double seed_sig_phi;  /* 0.001 rad, seed_sig_pt 0.01 (relative), seed_sig_z 0.05 cm: pixel-seed */
  double seed_sig_pt;   /*   resolutions used by pT3 / pT5 linking (C6)                           */
  double seed_sig_z;
  double sig_t[4];      /* precise (r-phi) hit resolution per category                            */
  double sig_z[4];      /* z resolution (barrel categories; 0 for endcap)                         */
  double sig_r[4];      /* r resolution (endcap categories; 0 for barrel)                         */
  int32_t dup_t5_shared;   /* 5: T5  duplicates share >= this many of 10 hits (S0)                */
  int32_t dup_pt5_shared;  /* 5: pT5 duplicates share >= this many OT hits   (S0)                 */
  int32_t dup_pt3_shared;  /* 3: pT3 duplicates share >= this many OT hits   (S0)                 */
  int32_t s0_enabled;      /* 1: intra-collection cleaning on                                     */
  uint32_t start_layer_mask; /* bit L set: an OT object whose first MD is in logical layer L may
                                be linked to a pixel seed (barrel L1,L2; disks 1,2 of both sides)  */
  /* capacities of the per-slot object arrays, as multiples of max_hits (MD, LS, T3, T5 and the
   * candidate counts that size the work lists) or of max_seeds (pT3, pT5).  Overflow is never
   * silent: lst_get_objects returns LST_ENOMEM for the slot. */
  float cap_md_per_hit, cap_ls_per_hit, cap_t3_per_hit, cap_t5_per_hit;
  float cap_pt3_per_seed, cap_pt5_per_seed;
  float cap_mdcand_per_hit, cap_lscand_per_hit, cap_t3cand_per_hit, cap_t5cand_per_hit;
  int32_t use_cuda_graph;  /* 1: lst_run replays one captured CUDA graph per slot               */
  int32_t enum_pruning;    /* enumeration shortcuts that never change a result (tests compare with 0):
                              bit 0: lst_create drops the module-map edges whose two lower-sensor boxes
                                     cannot hold a line segment (uses the boxes of lst_geometry);
                              bit 1: the LS pre-filter visits, per inner MD and connected module, only
                                     the MDs inside the azimuthal window / pointing cone that the cuts
                                     allow (uses the event's own MD positions only).  Default 3.      */
  int32_t use_pdl;         /* 1: every kernel of the chain but the first is launched with programmatic
                              stream serialisation (programmatic dependent launch): its blocks may become
                              resident while the preceding kernel drains; results are identical          */
  int32_t batch_events;    /* E in [1, 8], default 1: slots are grouped E at a time (group g = slots
                              [g E, (g + 1) E)) and lst_run_batch runs a whole group as ONE chain of
                              launches with a grid over (event, work): SURVEY.md 8(f)1, the B200 form of
                              the paper's multi-streaming                             */
  uint32_t trunc_cap[6][16]; /* occupancy truncation, default all 0 = exact:
                              trunc_cap[level][L] = K > 0: a module of logical layer L keeps at most K
                              objects of `level` (LST_MD .. LST_T5; an object belongs to the module of its
                              first mini-doublet); trunc_cap[LST_PT3 / LST_PT5][0] = K: a pixel seed keeps
                              at most K pT3 / pT5.  Kept are the K first in the canonical order of the
                              level (hits of a sensor ascend in azimuth relative to the module centre,
                              ties by caller index; candidates row-major over (left object, right object)).
                              The cap_* factors above can then be sized from the truncated occupancies
                              (paper_2209_13711_b200/occupancy.py).  The mode bounds what a BUCKET keeps, not the
                              slot's memory: the capacities stay global (cap_* x max_hits) and the work lists hold
                              the untruncated pre-filter survivors, so an event busier than the capacities allow
                              is still refused with LST_ENOMEM (never a silently smaller result); size them on a
                              sample that is disjoint from, and as busy as, the events to be served. */
  int32_t store_half;      /* 0 (default) | 1: reduced-precision storage (PAPER.md:147 outlook):
                              the derived floats that no later decision reads (MD dphi; LS dphi, kappa,
                              sigma_kappa; T3 beta; T5 R, chi2, kappa3 a / b, pT) are kept as IEEE binary16
                              in the slot workspace (half the bytes; relative error <= 4.9e-4, absolute 3e-8 for
                              magnitudes below 6.1e-5 such as the sigma_kappa of an LS, values above 65504 saturate) and widened again by lst_get_objects.  Object sets, keep flags
                              and the TC list are unchanged: every decision uses the fp64 quantities. */
  int32_t s0_fixpoint_passes; /* 0 (default): the non-greedy cleaning rule S0 (an object is removed iff SOME
                              better duplicate exists).  P = 2, 4, .. 16: S0 of the T5 collection is iterated
                              P more times towards the greedy fix-point "kept iff no KEPT better duplicate"
                              (cleaning of PAPER.md:77-83), which keeps every T5 the non-greedy
                              rule keeps plus those that lost only to removed objects.  After an even number of
                              passes the kept set is a duplicate-free subset of the fix-point, equal to it when
                              lst_get_fixpoint_unsettled reports 0 (8 passes on the 6 000-particle, 12 on the 13 500-particle synthetic events). */
} lst_config;

/* Detector description, HOST arrays of length n_modules (copied by the callee).  A module is a
 * two-sensor "pT module"; the box is that of its LOWER sensor (nearer the
 * origin).  Hit det ids are det = 2*module + sensor, sensor 0 = lower, 1 = upper.
 * PRECONDITION, checked for every event on the device: each lower-sensor hit lies inside its
 * module's box (tolerance 5e-5 cm in r and z, 4e-6 rad in azimuth).  lst_create's dead-edge pruning
 * and the pixel-seed windows are conservative interval arithmetic ON THESE BOXES, so a hit outside
 * would silently lose objects: such an event is rejected with LST_EINVAL instead.
 * lst_create / lst_build_module_map return LST_EINVAL unless 0 < rmin <= rmax, zmin <= zmax (equal
 * and non-zero for endcap categories: the sensor plane), 0 < half_phi <= 0.6 rad, |phic| <= 2 pi. */
typedef struct {
  uint32_t n_modules;
  const uint8_t *category;       /* 0 bPS, 1 b2S, 2 ePS, 3 e2S                                   */
  const uint8_t *logical_layer;  /* 0-5 barrel L1-6, 6-10 disks +z, 11-15 disks -z               */
  const float *rmin, *rmax;      /* radial extent                                                */
  const float *phic, *half_phi;  /* centre azimuth and half opening angle                        */
  const float *zmin, *zmax;      /* z extent (equal for endcap modules: the sensor plane)        */
} lst_geometry;

/* Module map (Fig. 4) in CSR form, HOST arrays: for module A, the connected
 * modules are cols[row_offsets[A] .. row_offsets[A+1]), ascending. */
typedef struct {
  const uint32_t *row_offsets;   /* n_modules + 1 */
  const uint32_t *cols;          /* row_offsets[n_modules] */
} lst_module_map;

/* One event's outer-tracker hits as SoA.  on_device = 0: HOST arrays (pinned
 * memory makes the upload asynchronous); 1: DEVICE arrays.  Borrowed only during the call to
 * lst_load_event itself (they are copied into the slot on the given stream; for HOST arrays the
 * caller must not modify them until that stream has passed the copy). */
typedef struct {
  uint32_t n;
  const float *x, *y, *z;
  const uint32_t *det;
  int on_device;
} lst_hits;

/* Pixel line segments (pLS): helix parameters + 4 pixel-hit ids (own id space). */
typedef struct {
  uint32_t n;
  const float *pt, *eta, *phi, *z0;
  const int8_t *q;
  const uint32_t *hit_ids;       /* 4*n */
  int on_device;
} lst_pixel_seeds;

/* A view of one object collection.  Pointers are DEVICE pointers into the slot workspace
 * (copy_to_host = 0) or HOST pointers into library-owned pinned staging (copy_to_host = 1);
 * both stay valid until the next lst_load_event or lst_get_objects (ANY level: the staging is one
 * buffer per slot) on the slot.
 *   hit_idx : n*arity ORIGINAL caller hit indices in layer order, lower hit before upper hit
 *             (arity: MD 2, LS 4, T3 6, T5 10, PT3 6, PT5 10, TC 14 = 10 OT (0xFFFFFFFF padded)
 *             + 4 pixel-hit ids (0xFFFFFFFF if none))
 *   parents : n*2: MD {module, 0}; LS {md_in, md_out}; T3 {ls_a, ls_b}; T5 {t3_a, t3_b};
 *             PT3 / PT5 {pls, t3 / t5}; TC {type (lst_level of the object; LST_TC = bare pLS), obj}
 *   f       : n*4 fp32: MD {dphi, kappa, sigma_kappa, 0}; LS {dphi, kappa, sigma_kappa, 0};
 *             T3 {beta, kappa3, sigma_kappa3, 0}; T5 {R, chi2, kappa3(1,2,3), kappa3(3,4,5)};
 *             PT3 / PT5 {chi2_pix, 0, 0, 0}; TC {pt, eta, phi, type}
 *   keep    : n bytes, T5 / PT3 / PT5 only: 1 = survives duplicate removal S0-S3 (else NULL) */
typedef struct {
  uint32_t n;
  uint32_t arity;
  const uint32_t *hit_idx;
  const uint32_t *parents;
  const float *f;
  const uint8_t *keep;
  int on_device;
} lst_objects;

typedef struct lst_ctx lst_ctx;

/* Fill *cfg with the defaults of DESIGN.md / SURVEY.md Appendix B. */
void lst_default_config(lst_config *cfg);

/* C2: module map of a detector = modules in the next logical layers reachable by
 * +-charged helices from the luminous region at the pT threshold (interval version, DESIGN.md
 * reading C2).  HOST only.  On success *row_offsets (n_modules+1) and *cols are malloc'd arrays
 * the caller frees with lst_free(). */
int lst_build_module_map(const lst_geometry *geom, const lst_config *cfg /* NULL = defaults */,
                         uint32_t **row_offsets, uint32_t **cols);
void lst_free(void *p);

/* Create a context on the current CUDA device: validates and uploads geometry + map (the host
 * arrays may be freed afterwards).  max_hits / max_seeds bound every event of every slot.
 * LST_EINVAL: null / empty / inconsistent geometry (see lst_geometry), category > 3, layer > 15, map
 * rows not ascending, column out of range, map degree > 512, or capacities (lst_config.cap_* x
 * max_hits / max_seeds) beyond the 32-bit candidate keys (roughly max_hits > 4 M with the defaults). */
int lst_create(const lst_geometry *geom, const lst_module_map *map, const lst_config *cfg /* NULL */,
               uint32_t n_slots, uint32_t max_hits, uint32_t max_seeds, lst_ctx **out);
void lst_destroy(lst_ctx *ctx);

/* Bytes of DEVICE workspace one slot needs (same for every slot). */
size_t lst_workspace_bytes(const lst_ctx *ctx);
/* Give slot `slot` its workspace: DEVICE memory, 256-byte aligned, >= lst_workspace_bytes(), owned
 * by the caller and borrowed until lst_destroy or the next bind.  LST_ENOMEM if too small.  With
 * lst_config.use_cuda_graph the slot's chain is captured and instantiated here; besides lst_create this
 * is the call that allocates (the graph, a small pinned header) and synchronises; lst_run only replays
 * the graph.  The one later allocation is the pinned staging of lst_get_objects(copy_to_host = 1), see
 * there. */
int lst_bind_workspace(lst_ctx *ctx, uint32_t slot, void *workspace, size_t bytes);

/* a0: copy one event into the slot (async on `cuda_stream`, a cudaStream_t passed as void*).
 * seeds may be NULL (no pixel seeds: pT3 / pT5 are empty, TC = cleaned T5).
 * LST_EINVAL: n > max_hits / max_seeds, null array with n > 0.  The event's CONTENT is checked on the
 * device by lst_run (det < 2 n_modules; x, y, z and the seed parameters finite; lower-sensor hits
 * inside their module's box); a violation makes lst_get_objects / lst_get_counts return LST_EINVAL
 * (lst_strerror names which), never a silently different result. */
int lst_load_event(lst_ctx *ctx, uint32_t slot, const lst_hits *hits, const lst_pixel_seeds *seeds,
                   void *cuda_stream);

/* a0-a6: enqueue the whole chain (index hits by det, MD, LS, T3, T5, pT5, pT3, S0-S3, TC) on
 * `cuda_stream`.  No host synchronisation; no allocation.  Sizes stay on the device. */
int lst_run(lst_ctx *ctx, uint32_t slot, void *cuda_stream);

/* The same chain for all the slots of group `group` (lst_config.batch_events consecutive slots, every
 * one of them bound and loaded, normally on this same stream) in ONE sequence of launches whose grids
 * span (event, work); with batch_events = 1 it is lst_run(group).  Results per slot are those of
 * lst_run.  LST_ESTATE if a slot of the group has no workspace or no event. */
int lst_run_batch(lst_ctx *ctx, uint32_t group, void *cuda_stream);
uint32_t lst_batch_events(const lst_ctx *ctx);

/* Number of T5 whose keep flag still changed in the last fix-point pass of the slot's last run
 * (lst_config.s0_fixpoint_passes > 0); 0 = the greedy fix-point was reached exactly. */
int lst_get_fixpoint_unsettled(lst_ctx *ctx, uint32_t slot, uint32_t *n_unsettled);

/* Synchronise the slot's stream and return a view of one level.  LST_ENOMEM if a collection
 * overflowed its capacity, LST_EINVAL if the event was invalid (see lst_load_event).
 * Allocation: copy_to_host = 0 allocates nothing.  The FIRST copy_to_host = 1 call on a slot allocates
 * that slot's pinned host staging (cudaMallocHost, sized for the largest level; kept until lst_destroy),
 * so slots that only hand out device views never pay for it: make that first call during warm-up if the
 * steady state must be allocation-free. */
int lst_get_objects(lst_ctx *ctx, uint32_t slot, lst_level level, int copy_to_host, lst_objects *out);

/* Per-level object counts of the slot's last run (synchronises); counts: uint32[LST_NLEVEL], HOST.
 * Also cheap way to wait for a slot.  cand (optional, may be NULL; uint64[18]), each in the order
 * MD, LS, T3, T5, pT5, pT3: [0..5] the candidates of the method's definition (e.g. LS: all MD pairs
 * in map-connected modules), [6..11] those that survived the stage's fp32 pre-filter and were
 * decided in fp64, [12..17] those the pre-filter kernel actually evaluated (fewer than [0..5] where
 * the enumeration is restricted to a window, see lst_config.enum_pruning). */
int lst_get_counts(lst_ctx *ctx, uint32_t slot, uint32_t *counts, uint64_t *cand);

/* Number of kernels the last lst_run / lst_run_timed of this context enqueued (or captured into
 * its graph); 0 before the first run.  For launch accounting in benchmarks. */
uint32_t lst_launches_per_run(const lst_ctx *ctx);

/* Measurement aid (per-kernel ms): the same chain as lst_run, launched without a
 * CUDA graph with one CUDA event after every kernel, then synchronised.  names[k] (HOST array of
 * max_kernels pointers to static strings, may be NULL) and ms[k] (HOST, may be NULL) receive the
 * kernel name and its duration on the stream (launch gap included); *n_kernels the number of
 * kernels in the chain (may exceed max_kernels; only max_kernels entries are written).
 * The objects it leaves in the slot are those of lst_run. */
int lst_run_timed(lst_ctx *ctx, uint32_t slot, void *cuda_stream, uint32_t max_kernels, const char **names,
                  float *ms, uint32_t *n_kernels);

const char *lst_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif
