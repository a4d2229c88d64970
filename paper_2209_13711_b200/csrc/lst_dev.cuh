// lst_dev.cuh -- device-side data layout and the work-item machinery shared by all stage kernels.
//
// Every stage (MD, LS, T3, T5, pT5, pT3) is a join: rows x per-row candidate lists, grouped so
// that one group's operands fit in shared memory.  A stage is FIVE launches:
//   groups  : per group g, rows R_g and candidates per row (uniform W_g, or a per-row list); the
//             group's candidates are cut into work ITEMS of <= 1024 candidates (one pass bit each);
//             the last block to finish scans the per-block item counts (first item of every group)
//   eval    : fp32 pre-filter on every candidate; the survivors (item, candidate, pair) are
//             appended to the stage's candidate list through warp-private staging
//   decide  : one thread per listed candidate: fp64 decision, pass BIT of the candidate, the
//             computed quantities into the pool at the candidate's list index
//   counts  : per-item pass counts and word prefixes from the pass bits; per-block sums, the last
//             block to finish scans them (exact sizes, no truncation)
//   fill    : one thread per listed candidate: the accepted ones move to item_base + bit rank; the
//             same kernel derives the level's CSR by first constituent from the ranks
// Output order is canonical (ascending item, ascending candidate) whatever order the list was
// appended in; warp ballots / prefix sums do the compaction, the atomics only order scratch lists.
// Every kernel takes a BATCH of slots (events) and picks its own with blockIdx.z: one chain of
// launches serves up to kMaxBatch events, and every kernel starts with
// griddepcontrol.wait so that the chain can be launched with programmatic dependent launch.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "lst_math.cuh"

namespace lst {

constexpr int kItemCand = 1024;          // candidates per work item
constexpr int kItemWords = kItemCand / 32;
constexpr int kThreads = 128;            // threads per block of eval / fill kernels
constexpr int kMaxRpi = 128;             // max rows per item
constexpr int kMaxBatch = 8;             // events (slots) one chain of launches can serve
constexpr int kMaxFixPasses = 16;        // lst_config.s0_fixpoint_passes (even, <= this)
constexpr int kRowChunk = 128;           // rows per group in the variable-width stages (T3, T5, pixel)
constexpr int kMaxDeg = 512;             // maximum module-map degree (checked by lst_create)
constexpr int kPxCap = 64;               // (seed, start module) rows per pixel seed ON AVERAGE (overflow -> LST_ENOMEM)
constexpr int kAdjCap = 32;              // related pixel seeds per pixel seed (overflow -> LST_ENOMEM)
constexpr int kEtaBins = 2048;           // eta bins of the pixel-seed lookup used by the cleaning
constexpr int kScanBlocks = 128;         // blocks of the two-pass device-wide scan
constexpr int kCountBlocks = 148;        // blocks of k_counts (per-item pass counts + two-level scan)
constexpr int kCountThreads = 512;
constexpr int kFlagBlocks = 592;         // blocks of k_s3_flags / k_tc_fill
constexpr int kScanThreads = 512;
constexpr int kPairLevel = 7;            // Header::n_obj slot that holds the (seed, module) pair count

enum Stage { S_MD = 0, S_LS, S_T3, S_T5, S_PT5, S_PT3, S_NSTAGE };

enum ErrBits {
  ERR_DET = 1u << 0,        // det id out of range
  ERR_CAP_ITEMS = 1u << 1,  // a work list overflowed
  ERR_CAP_OBJ = 1u << 2,    // an object array overflowed
  ERR_CAP_PIX = 1u << 3,    // a per-seed list (compatible modules / related seeds) overflowed
  ERR_NONFINITE = 1u << 4,  // a hit coordinate or a pixel-seed parameter is NaN or infinite
  ERR_BOX = 1u << 5         // a lower-sensor hit lies outside its module's box (lst_geometry)
};
constexpr float kBoxTolLen = 5e-5f;   // cm: half the growth the host-side box arithmetic allows for
constexpr float kBoxTolPhi = 5e-7f;   // rad (+ the fp32 rounding of the two azimuths, < 4e-6 in all)

// Item geometry of a group with R rows and W columns (MD, LS; a join group is one "row" of W flat
// candidates).  W <= kItemCand: one column tile, item_rpi(W) rows per item; else one row per item and
// ceil(W / kItemCand) column tiles.  Item (q, ct) of the group = g_item0 + q * n_ct + ct.
__host__ __device__ __forceinline__ uint32_t item_rpi(uint32_t W) {
  if (W > (uint32_t)kItemCand) return 1u;
  const uint32_t r = (uint32_t)kItemCand / W;
  return r > (uint32_t)kMaxRpi ? (uint32_t)kMaxRpi : r;
}
__host__ __device__ __forceinline__ uint32_t item_nct(uint32_t W) {
  return W <= (uint32_t)kItemCand ? 1u : (W + kItemCand - 1) / kItemCand;
}
// items of a group with R rows and W columns
__host__ __device__ __forceinline__ uint32_t items_of(uint32_t R, uint32_t W) {
  if (R == 0 || W == 0) return 0;
  const uint32_t rpi = item_rpi(W);
  return ((R + rpi - 1) / rpi) * item_nct(W);
}

// "last block" tickets of the kernels whose final block runs a small serial epilogue
enum Ticket { TK_HIST = 0, TK_GROUPS = 1 /* + stage */, TK_COUNTS = 7 /* + stage */, TK_SEEDS = 13, TK_FLAGS = 14, TK_N = 16 };

struct Header {          // per slot, device; everything after n_seeds is zeroed at the start of lst_run
  uint32_t n_hits, n_seeds;
  uint32_t n_obj[8];                 // indexed by lst_level; [kPairLevel] = (seed, module) pairs
  uint32_t n_items[S_NSTAGE];
  uint32_t n_groups[S_NSTAGE];
  uint32_t next_unit[S_NSTAGE];      // dynamic work distribution: next row block to hand out
  uint32_t cl_used[S_NSTAGE];        // pre-filter survivors appended to the stage's candidate list
  uint32_t err;
  uint32_t n_inc;                    // 3 * n_hits: rows of the (hit, object type) -> objects incidence
  uint32_t n_heavy[kMaxFixPasses + 1];     // per S0 pass: objects k_s0 handed to k_s0_heavy (listed in tc_pos, free until S3)
  uint32_t heavy_next[kMaxFixPasses + 1];  // ... and the next one to hand out
  uint32_t n_unsettled;              // T5 whose flag still changed in the last fix-point pass (0: the fix-point was reached)
  uint32_t flag_chunk;               // keep flags per block of k_s3_flags / k_tc_fill
  uint32_t ticket[TK_N];             // blocks that finished (last_block)
  unsigned long long cand[S_NSTAGE]; // candidates of the method's definition per stage (rows x connected columns)
  unsigned long long cand_eval[S_NSTAGE];   // candidates the stage's pre-filter kernel actually evaluated
};

struct StageBuf {        // work list of one stage
  uint32_t *gR, *gW;     // [cap_groups] rows / width (or candidate count) per group
  uint32_t *g_item0;     // [cap_groups+1] first item of a group
  uint32_t *gblk;        // [cap_groups / groups per block + 2] items of the groups of one block of the groups kernel
  uint32_t *item_group;  // [cap_items] group of an item (MD only: the module)
  uint32_t *row_start, *row_cum;   // [cap_rows] joins: first right object of a row / candidates of the group before the row
  uint32_t *cblk;        // [kCountBlocks + 1] pass counts of the items of one block of k_counts
  uint32_t *mask;        // [cap_items * kItemWords]
  uint16_t *wpre;        // [cap_items * kItemWords] pass count of the item's words before this one
  uint32_t *item_cnt;    // [cap_items] pass count
  uint32_t *item_base;   // [cap_items] exclusive prefix
  // pool: what the decide kernel computed for accepted candidate j of the candidate list (same
  // index j: no counter, no atomics); the fill kernel moves the entries whose pass bit is set to their
  // canonical position item_base[item] + rank of the candidate
  double2 *p_d2, *p_d2b; // [cap_cl] fp64 results (p_d2b: T5 only)
  float4 *p_f4;          // [cap_cl] fp32 results
  // candidate list: survivors of the cheap pre-filter kernel, decided in fp64 by the decide kernel
  uint32_t *cl_key;      // [cap_cl] item * kItemCand + candidate
  uint2 *cl_ab;          // [cap_cl] the pair (row object, column object)
  uint32_t cap_groups, cap_items, cap_pool, cap_cl;
};

// Per module and event (k_ls_groups): everything a row of the LS pre-filter needs about the MDs of a
// connected module, in one 64-byte record: the bounding box of their anchors, their first index and
// count, and where their azimuth keys (md_prel, ascending) cross 14 equidistant edges between the
// smallest and the largest key, so that an azimuthal window becomes an index range with no search.
constexpr int kModBins = 15;
struct __align__(16) ModEv {
  float rlo, rhi, zlo, zhi;        // anchors: rt and z extent
  float pmin, inv_w, phic;         // smallest key, bins per radian (0: no bin table), the module's centre azimuth
  uint32_t first;                  // index of the module's first MD
  uint32_t n_cat;                  // MDs in the module | category << 30
  uint16_t cum[kModBins - 1];      // cum[j] = MDs with key < pmin + (j + 1) / inv_w
};
static_assert(sizeof(ModEv) == 64, "ModEv is one 64-byte record");

// Static detector data (device), shared by all slots.
struct GeoDev {
  uint32_t n_modules, n_det;
  const uint8_t *category, *layer;
  const uint32_t *map_off, *map_cols;
  // boxes of the lower sensors (lst_geometry) and the modules that may start a pT3 / pT5 (C6)
  const float *rmin, *rmax, *phic, *hphi, *zmin, *zmax;
  const uint32_t *start_mods;
  uint32_t n_start;
  // start modules grouped into "rows": modules that differ only in phic (same category, r, z and
  // half_phi box, e.g. one z-row of a barrel layer or one ring of a disk).  prow_b1 = {hphi, rmin,
  // rmax, category}, prow_b2 = {zmin, zmax, sig_t / rmin, 0}; members prow_off[r] .. prow_off[r+1]:
  // prow_k = index into start_mods, prow_phic = its phic.
  const float4 *prow_b1, *prow_b2;
  const uint32_t *prow_off, *prow_k;
  const float *prow_phic;
  const uint32_t *prow_of;   // [n_start] row of start module k
  uint32_t n_prow;
};

// All per-slot arrays (device pointers into the caller's workspace).
struct SlotDev {
  Header *hdr;
  // raw event
  float *raw_x, *raw_y, *raw_z; uint32_t *raw_det;
  float *seed_pt, *seed_eta, *seed_phi, *seed_z0; int8_t *seed_q; uint32_t *seed_ids;
  // a0: hits grouped by det
  uint32_t *det_cnt, *det_off;               // [n_det+1]
  uint32_t *md_row0;                         // [n_modules+1] lower-sensor hits (rows of the MD stage) of the modules before m
  uint32_t *row_mod;                         // [cap_hits] module of MD row t (t-th lower-sensor hit in sorted order)
  uint32_t *tmp_slot;                        // [cap_hits] arrival rank of a hit inside its det (k_hist)
  uint32_t *tmp_orig;                        // [cap_hits]
  float *tmp_key, *hit_key;                  // [cap_hits] azimuth relative to the module centre (sort key inside a det)
  float4 *hit;                               // [cap_hits] x, y, z, rt
  uint32_t *hit_orig;                        // [cap_hits] original caller index
  // MD
  float4 *md_pos;        // anchor (lower hit) x, y, z, rt
  double2 *md_kd;        // kappa_MD, sigma_kappa_MD (fp64: they enter the LS decision)
  float2 *md_kf;         // same, fp32 (pre-filter)
  uint2 *md_hit;         // sorted positions of lower / upper hit
  uint32_t *md_mod;      // module << 2 | category
  float *md_dphi;
  float *md_phi;         // azimuth of the anchor, fp32 (pixel-linking pre-filter)
  float *md_prel;        // the anchor's sort key (azimuth relative to the module centre): ascending inside a module
  uint32_t *md_mod_off;  // [n_modules+1]
  ModEv *mod_ev;         // [n_modules] what the LS enumeration needs to know about a module's MDs in this event
  uint32_t *edge_col0;   // [map edges] column of module A's candidate rectangle where the MDs of cols[e] start
  // LS
  uint2 *ls_md;          // inner, outer MD
  float4 *ls_f;          // dphi, kappa, sigma_kappa, 0
  uint32_t *ls_md_off;   // [cap_md+1] LS range of an inner MD
  // T3
  uint4 *t3_md;          // md1, md2, md3, 0
  uint2 *t3_ls;
  double2 *t3_kd;        // kappa3, sigma_kappa3
  float *t3_beta;
  uint32_t *t3_md_off;   // [cap_md+1] T3 range of a first MD
  // T5
  uint32_t *t5_md;       // [5 * cap_t5]
  uint2 *t5_t3;
  double *t5_chi2;
  double2 *t5_etaphi;
  float4 *t5_f;          // R, chi2, k3a, k3b
  float *t5_pt;
  uint8_t *t5_keep;
  uint8_t *t5_keep2;     // second flag buffer of the S0 fix-point passes
  uint32_t *t5_md_off;   // [cap_md+1] T5 range of a first MD
  // pixel-seeded
  uint2 *pt5_po, *pt3_po;          // pls, obj
  double *pt5_chi2, *pt3_chi2;
  uint8_t *pt5_keep, *pt3_keep, *pls_keep;
  uint32_t *px_cnt;                // [cap_seeds] compatible start modules of a seed
  uint32_t *px_bits;               // [cap_seeds * ceil(n_start / 32)] one bit per (seed, start module)
  uint32_t *px_off;                // [cap_seeds+1]
  uint2 *px_pair;                  // [cap_seeds * kPxCap] (seed, module), ascending: rows of the pixel joins
  uint2 *px_rng;                   // [cap_seeds * kPxCap] the row's MDs: those of its module inside the seed's azimuthal window
  uint32_t *pt5_pls_off, *pt3_pls_off;   // [cap_seeds+1] pT5 / pT3 range of a seed
  // a6 cleaning
  uint32_t *t5_hits, *pt3_hits;    // [10 cap_t5], [6 cap_pt3] sorted hit positions in layer order
  uint32_t *inc_cnt, *inc_cur;     // [3 cap_hits+1] each, contiguous: (hit, type) -> objects incidence, row 3 h + type
  uint32_t *inc_off;               // [3 cap_hits+1]
  uint32_t *inc_ent;               // [10 cap_t5 + 10 cap_pt5 + 6 cap_pt3] object ids (T5 | pT5 | pT3)
  uint32_t *pls_bin_cnt, *pls_bin_cur;   // [kEtaBins] each (zeroed per run): seeds per eta bin, fill cursor
  uint32_t *pls_bin_off;           // [kEtaBins+1]
  uint32_t *pls_bin_ent;           // [cap_seeds]
  uint32_t *pls_adj_cnt, *pls_adj; // [cap_seeds], [cap_seeds * kAdjCap]: seeds close in eta-phi to a seed
  // pixel-hit ids: open-addressing hash set (key = 1 << 32 | id, 0 = empty), the slot of each of a
  // seed's 4 ids, and per slot "some surviving pT5 / pT3 uses a seed with this pixel hit"
  unsigned long long *pid_key;     // [pid_size]
  uint32_t *pls_slot;              // [4 * cap_seeds]
  uint8_t *pid_has5, *pid_has3;    // [pid_size] each, contiguous
  uint32_t pid_size;               // power of two >= 8 * cap_seeds
  uint8_t *pls_has5, *pls_has3, *pls_near_t5;   // [cap_seeds] each, contiguous
  unsigned long long *pls_min5, *pls_min3;      // [cap_seeds] bit pattern of the seed's minimum pT5 / pT3 score
  uint32_t *pls_best5, *pls_best3;              // [cap_seeds] the seed's best pT5 / pT3 (index in its collection), or ~0
                                                // (the four arrays are contiguous: one memset)
  uint8_t *hit_used5, *hit_used3;  // [cap_hits] each, contiguous: hit belongs to a surviving pT5 / pT3 (S1, S2)
  uint32_t *tc_flag, *tc_pos;      // [cap_tc+1] keep flags in TC order; tc_pos: the objects k_s0 hands to k_s0_heavy
  uint32_t *flag_blk;              // [kFlagBlocks+1] kept flags per block of k_s3_flags, then their exclusive prefix
  uint32_t *scan_part;             // [kScanBlocks+2]: block partials, total; last word = ticket
  // TC
  uint2 *tc_to;                    // type, obj
  float4 *tc_f;                    // pt, eta, phi, type
  // work lists
  StageBuf st[S_NSTAGE];
  uint32_t cap_hits, cap_seeds, cap_md, cap_ls, cap_t3, cap_t5, cap_pt3, cap_pt5, cap_tc;
  // export scratch
  uint32_t *exp_hits, *exp_par; float *exp_f;
  // lst_config.store_half: the derived floats that no later decision reads
  // (md_dphi, ls_f, t3_beta, t5_f, t5_pt) are stored as IEEE binary16; the arrays above then hold 2-byte
  // elements (same pointers, half the bytes) and are accessed through ld_f / st_f / ld_f4 / st_f4
  uint32_t half_store;
};

// A derived float (or float4) at index i of an array that holds fp32 or, with half_store, binary16 elements
// (round to nearest; |v| above the binary16 range saturates to +-65504 instead of becoming infinite).
__device__ __forceinline__ __half to_half_sat(float v) { return __float2half_rn(fminf(65504.0f, fmaxf(-65504.0f, v))); }
__device__ __forceinline__ void st_f(const SlotDev &s, float *arr, size_t i, float v) {
  if (s.half_store) reinterpret_cast<__half *>(arr)[i] = to_half_sat(v); else arr[i] = v;
}
__device__ __forceinline__ float ld_f(const SlotDev &s, const float *arr, size_t i) {
  return s.half_store ? __half2float(reinterpret_cast<const __half *>(arr)[i]) : arr[i];
}
__device__ __forceinline__ void st_f4(const SlotDev &s, float4 *arr, size_t i, float4 v) {
  if (s.half_store) {
    const __half2 a = __halves2half2(to_half_sat(v.x), to_half_sat(v.y)), b = __halves2half2(to_half_sat(v.z), to_half_sat(v.w));
    reinterpret_cast<uint2 *>(arr)[i] = make_uint2(*reinterpret_cast<const uint32_t *>(&a), *reinterpret_cast<const uint32_t *>(&b));
  } else arr[i] = v;
}
__device__ __forceinline__ float4 ld_f4(const SlotDev &s, const float4 *arr, size_t i) {
  if (!s.half_store) return arr[i];
  const uint2 u = reinterpret_cast<const uint2 *>(arr)[i];
  const float2 a = __half22float2(*reinterpret_cast<const __half2 *>(&u.x)), b = __half22float2(*reinterpret_cast<const __half2 *>(&u.y));
  return make_float4(a.x, a.y, b.x, b.y);
}

// The slots (events) one chain of launches serves: a kernel's blocks with blockIdx.z = e work on
// slot s[e].  Passed by value as a __grid_constant__ kernel parameter (CUDA >= 12.1 allows 32 KB).
struct Batch {
  SlotDev s[kMaxBatch];
};
#define LST_SLOT(B) const SlotDev &s = (B).s[blockIdx.z]

// ------------------------------------------------------------------ programmatic dependent launch
// Every kernel of the chain calls pdl_enter() before it touches memory: griddepcontrol.wait blocks
// until the preceding kernel of the stream has completed and its writes are visible (a no-op when
// the kernel was launched without the programmatic-serialisation attribute).  No kernel triggers its
// dependents early (griddepcontrol.launch_dependents): a dependent's blocks would take SM slots from
// blocks of this kernel that have not started yet (measured: slower); the implicit trigger at block
// exit lets the next kernel's launch overlap this kernel's tail and its memory flush.
__device__ __forceinline__ void pdl_enter() {
#if defined(__CUDA_ARCH__)
  asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
}

// ------------------------------------------------------------------ small device helpers
__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ uint32_t warp_excl_scan(uint32_t v, uint32_t *total) {
  const int lane = threadIdx.x & 31;
  uint32_t x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  *total = __shfl_sync(0xffffffffu, x, 31);
  return x - v;
}

// Block-wide exclusive scan of one value per thread (blockDim.x <= 1024); sh: 33 words.
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t *sh, uint32_t *total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  uint32_t wt;
  uint32_t e = warp_excl_scan(v, &wt);
  __syncthreads();
  if (lane == 0) sh[w] = wt;
  __syncthreads();
  if (w == 0) {
    uint32_t t = lane < nw ? sh[lane] : 0, tt;
    uint32_t ee = warp_excl_scan(t, &tt);
    sh[lane] = ee;
    if (lane == 0) sh[32] = tt;
  }
  __syncthreads();
  e += sh[w];
  *total = sh[32];
  return e;
}

// "Last block" epilogue: every block calls this after its last global write; exactly one block
// (the last to arrive) gets true, after which it sees the writes of all the others (read them with
// __ldcg: L1 is not coherent).  ticket: a zeroed word of the slot header; nblocks = blocks that call.
__device__ __forceinline__ bool last_block(uint32_t *ticket, uint32_t nblocks) {
  __shared__ bool lb_last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) lb_last = atomicAdd(ticket, 1u) == nblocks - 1u;
  __syncthreads();
  const bool l = lb_last;
  if (l) __threadfence();
  return l;
}

// Last-block scan used by the groups kernels and k_counts: exclusive scan of part[0 .. n) in place
// (n <= a few thousand), total returned to every thread.  sh: 33 words.
__device__ __forceinline__ uint32_t lb_scan_parts(uint32_t *part, uint32_t n, uint32_t *sh) {
  const uint32_t chunk = (n + blockDim.x - 1) / blockDim.x;
  const uint32_t b0 = min(n, threadIdx.x * chunk), b1 = min(n, b0 + chunk);
  uint32_t sum = 0;
  for (uint32_t i = b0; i < b1; ++i) sum += __ldcg(&part[i]);
  uint32_t tot;
  uint32_t run = block_excl_scan(sum, sh, &tot);
  for (uint32_t i = b0; i < b1; ++i) { const uint32_t v = __ldcg(&part[i]); part[i] = run; run += v; }
  __syncthreads();
  return tot;
}

// Exclusive scan of in[0..n) into out[0..n], out[n] = total; one block, in and out 16-byte aligned.
// Coalesced: per round thread t owns the four elements 4 (round * blockDim.x + t) .. + 3 (one uint4
// load, one block scan, one uint4 store).  The input was written by other blocks of the same kernel
// (last-block epilogue): read through L2.
__device__ __forceinline__ void block_scan_array(const uint32_t *in, uint32_t *out, uint32_t n, uint32_t *sh) {
  uint32_t carry = 0;
  for (uint32_t base = 0; base < n; base += 4 * blockDim.x) {
    const uint32_t i = base + 4 * threadIdx.x;
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (i + 3 < n) v = __ldcg(reinterpret_cast<const uint4 *>(in + i));
    else {
      if (i < n) v.x = __ldcg(&in[i]);
      if (i + 1 < n) v.y = __ldcg(&in[i + 1]);
      if (i + 2 < n) v.z = __ldcg(&in[i + 2]);
    }
    uint32_t tot;
    const uint32_t e = carry + block_excl_scan(v.x + v.y + v.z + v.w, sh, &tot);
    const uint4 o = make_uint4(e, e + v.x, e + v.x + v.y, e + v.x + v.y + v.z);
    if (i + 3 < n) *reinterpret_cast<uint4 *>(out + i) = o;
    else {
      if (i < n) out[i] = o.x;
      if (i + 1 < n) out[i + 1] = o.y;
      if (i + 2 < n) out[i + 2] = o.z;
    }
    carry += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) out[n] = carry;
}

// Last-block epilogue of the two-level scans: arr[i] += blk[i / per_block] for i < n (arr holds the
// exclusive prefix inside its block, blk the exclusive prefix of the block sums).  Four independent
// loads in flight per thread (the values come from other blocks: read through L2).
__device__ __forceinline__ void lb_add_block_prefix(uint32_t *arr, uint32_t n, const uint32_t *blk, uint32_t per_block) {
  if (per_block == 0) return;
  const uint32_t T = blockDim.x;
  for (uint32_t base = threadIdx.x; base < n; base += 4 * T) {
    uint32_t v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) { const uint32_t i = base + k * T; v[k] = i < n ? __ldcg(&arr[i]) + blk[i / per_block] : 0u; }
#pragma unroll
    for (int k = 0; k < 4; ++k) { const uint32_t i = base + k * T; if (i < n) arr[i] = v[k]; }
  }
}

// eta bins of the pixel seeds ("close in eta-phi" lookups of the cleaning, reading C7)
__device__ __forceinline__ int eta_bin(const Params &g, double eta) {
  const double t = (eta + 4.0) * g.eta_bin_inv;
  if (!(t >= 0.0)) return 0;
  return t < (double)g.eta_nbins ? (int)t : g.eta_nbins - 1;
}
__device__ __forceinline__ bool close_eta_phi(const Params &g, double e1, double p1, double e2, double p2) {
  const double de = e1 - e2;
  if (fabs(de) > g.dr_eta_pre) return false;
  const double dp = wrap_pi(p1 - p2);
  return de * de + dp * dp < g.dr2max;
}

// One warp: the seeds b != a close to seed a in eta-phi, found through the eta bins (a close seed
// lies in a's bin or a neighbouring one: the bin width exceeds sqrt(dr2max)).
__device__ __forceinline__ void pls_adjacent(const SlotDev &s, const Params &g, uint32_t a) {
  const int lane = threadIdx.x & 31;
  const double ea = (double)s.seed_eta[a], pa = (double)s.seed_phi[a];
  const int b0 = eta_bin(g, ea);
  const int lo = b0 > 0 ? b0 - 1 : 0, hi = b0 + 1 < g.eta_nbins ? b0 + 1 : g.eta_nbins - 1;
  const uint32_t e0 = s.pls_bin_off[lo], e1 = s.pls_bin_off[hi + 1];
  uint32_t cnt = 0;
  for (uint32_t eb = e0; eb < e1; eb += 32) {
    const uint32_t e = eb + lane;
    uint32_t b = 0;
    bool close = false;
    if (e < e1) {
      b = s.pls_bin_ent[e];
      close = b != a && close_eta_phi(g, ea, pa, (double)s.seed_eta[b], (double)s.seed_phi[b]);
    }
    const uint32_t bal = __ballot_sync(0xffffffffu, close);
    const uint32_t pos = cnt + __popc(bal & ((1u << lane) - 1u));
    if (close && pos < (uint32_t)kAdjCap) s.pls_adj[(size_t)a * kAdjCap + pos] = b;
    cnt += __popc(bal);
  }
  if (cnt > (uint32_t)kAdjCap) { if (lane == 0) atomicOr(&s.hdr->err, (uint32_t)ERR_CAP_PIX); cnt = 0; }
  if (lane == 0) s.pls_adj_cnt[a] = cnt;
}

// Warp-private ring queue (64 entries in shared memory; head / count are warp-uniform registers).
// A stage pushes its sparse survivors; the next stage pops them 32 at a time, so that the expensive
// arithmetic always runs on full warps and no block-wide barrier separates the stages.
struct WarpQueue {
  uint32_t *q;       // 64 words of shared memory owned by this warp
  uint32_t head, n;
  __device__ __forceinline__ void init(uint32_t *mem) { q = mem; head = 0; n = 0; }
  // all 32 lanes must call; at most 32 entries are added, the caller keeps n <= 32 before a push
  __device__ __forceinline__ void push(bool keep, uint32_t v) {
    const uint32_t b = __ballot_sync(0xffffffffu, keep);
    if (b == 0) return;
    const int lane = threadIdx.x & 31;
    if (keep) q[(head + n + __popc(b & ((1u << lane) - 1u))) & 63u] = v;
    n += __popc(b);
    __syncwarp();
  }
  // pops min(n, 32) entries: lane < count gets one (returns true)
  __device__ __forceinline__ bool pop(uint32_t *v) {
    const int lane = threadIdx.x & 31;
    const uint32_t take = n < 32u ? n : 32u;
    const bool have = (uint32_t)lane < take;
    *v = q[(head + lane) & 63u];
    __syncwarp();
    head = (head + take) & 63u;
    n -= take;
    return have;
  }
};

// The same with three words per entry (the LS pre-filter carries inner MD, outer MD and candidate key
// from tier 1 to tier 2 across row boundaries).
struct WarpQueue3 {
  uint32_t *q;       // 3 x 64 words of shared memory owned by this warp
  uint32_t head, n;
  __device__ __forceinline__ void init(uint32_t *mem) { q = mem; head = 0; n = 0; }
  __device__ __forceinline__ void push(bool keep, uint32_t a, uint32_t b, uint32_t c) {
    const uint32_t bal = __ballot_sync(0xffffffffu, keep);
    if (bal == 0) return;
    const int lane = threadIdx.x & 31;
    if (keep) {
      const uint32_t p = (head + n + __popc(bal & ((1u << lane) - 1u))) & 63u;
      q[p] = a; q[64 + p] = b; q[128 + p] = c;
    }
    n += __popc(bal);
    __syncwarp();
  }
  __device__ __forceinline__ bool pop(uint32_t *a, uint32_t *b, uint32_t *c) {
    const int lane = threadIdx.x & 31;
    const uint32_t take = n < 32u ? n : 32u;
    const bool have = (uint32_t)lane < take;
    const uint32_t p = (head + lane) & 63u;
    *a = q[p]; *b = q[64 + p]; *c = q[128 + p];
    __syncwarp();
    head = (head + take) & 63u;
    n -= take;
    return have;
  }
};

// eval epilogue, one warp: publish an item's mask words (lane = word), their running pass counts
// and the item's pass count.
__device__ __forceinline__ void publish_item(const StageBuf &st, uint32_t it, uint32_t w) {
  const int lane = threadIdx.x & 31;
  uint32_t tot;
  const uint32_t e = warp_excl_scan((uint32_t)__popc(w), &tot);
  st.mask[(size_t)it * kItemWords + lane] = w;
  st.wpre[(size_t)it * kItemWords + lane] = (uint16_t)e;
  if (lane == 0) st.item_cnt[it] = tot;
}

// Warp-private staging of candidate-list entries (ring in shared memory): the sparse survivors of
// many pre-filter iterations are appended BATCH at a time, i.e. one atomic on the list counter per
// BATCH entries (the counter is a single address: per-iteration atomics serialise in L2).
template <int BATCH>                 // 32 or 64; the ring holds BATCH + 32 .. 2 * BATCH entries
struct ClStageT {
  uint32_t key[2 * BATCH];
  uint2 ab[2 * BATCH];
};
template <int BATCH>
struct ClBufT {
  ClStageT<BATCH> *m;
  uint32_t head, n;
  static constexpr uint32_t kMask = 2 * BATCH - 1;
  __device__ __forceinline__ void init(ClStageT<BATCH> *mem) { m = mem; head = 0; n = 0; }
  // all 32 lanes call; flushes a full batch when one is ready
  __device__ __forceinline__ void push(Header *hdr, const StageBuf &st, int stage, bool keep, uint32_t key, uint2 ab) {
    const uint32_t b = __ballot_sync(0xffffffffu, keep);
    if (b == 0) return;
    const int lane = threadIdx.x & 31;
    if (keep) {
      const uint32_t p = (head + n + __popc(b & ((1u << lane) - 1u))) & kMask;
      m->key[p] = key; m->ab[p] = ab;
    }
    n += __popc(b);
    __syncwarp();
    if (n >= (uint32_t)BATCH) flush(hdr, st, stage);
  }
  __device__ __forceinline__ void flush(Header *hdr, const StageBuf &st, int stage) {
    const int lane = threadIdx.x & 31;
    const uint32_t take = n < (uint32_t)BATCH ? n : (uint32_t)BATCH;
    uint32_t base = 0;
    if (lane == 0) base = atomicAdd(&hdr->cl_used[stage], take);
    base = __shfl_sync(0xffffffffu, base, 0);
    for (uint32_t k = lane; k < take; k += 32) {
      const uint32_t p = (head + k) & kMask, pos = base + k;
      if (pos < st.cap_cl) { st.cl_key[pos] = m->key[p]; st.cl_ab[pos] = m->ab[p]; }
      else atomicOr(&hdr->err, (uint32_t)ERR_CAP_ITEMS);
    }
    __syncwarp();
    head = (head + take) & kMask;
    n -= take;
  }
  __device__ __forceinline__ void flush_all(Header *hdr, const StageBuf &st, int stage) {
    while (n) flush(hdr, st, stage);
  }
};
typedef ClStageT<32> ClStage;
typedef ClBufT<32> ClBuf;

// Number of accepted candidates with a key below `key` (= item * kItemCand + candidate): the canonical
// index at which the objects of a row start, given the key of the row's first candidate.  The masks
// are cleared item by item (all 32 words), so a key past the item's last candidate is fine.
__device__ __forceinline__ uint32_t rank_before(const StageBuf &st, uint32_t n_items, uint32_t n_total, uint32_t key) {
  const uint32_t it = key / (uint32_t)kItemCand, c = key % (uint32_t)kItemCand;
  if (it >= n_items) return n_total;
  const size_t w = (size_t)it * kItemWords + (c >> 5);
  return st.item_base[it] + st.wpre[w] + __popc(st.mask[w] & ((1u << (c & 31)) - 1u));
}

// fill: canonical index of listed candidate `key` = item * kItemCand + candidate, or 0xFFFFFFFF if
// the decide kernel did not accept it (its pass bit is clear)
__device__ __forceinline__ uint32_t pool_target(const StageBuf &st, uint32_t key) {
  const uint32_t it = key / (uint32_t)kItemCand, c = key % (uint32_t)kItemCand;
  const size_t w = (size_t)it * kItemWords + (c >> 5);
  const uint32_t m = st.mask[w];
  if (!((m >> (c & 31)) & 1u)) return 0xFFFFFFFFu;
  return st.item_base[it] + st.wpre[w] + __popc(m & ((1u << (c & 31)) - 1u));
}

}  // namespace lst
