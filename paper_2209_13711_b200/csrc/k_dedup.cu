// k_dedup.cu -- a6 duplicate removal and track candidates (reading C7, steps S0-S4).
//
// Every rule is non-greedy ("a is removed iff SOME b of the named set satisfies the condition"), so
// each object decides its own fate from read-only data: one thread per object, keep flags only,
// no ordering between threads.  Pairs are found through two lookups instead of all-pairs loops:
//   * hit -> objects incidence lists (CSR over the sorted hit positions) for "shares OT hits";
//   * pixel seeds binned in eta (bin width >= 1.25 sqrt(dr2max)) for "close in eta-phi", plus a
//     per-seed list of the seeds close to it; a hash set of the pixel-hit ids for "shares a pixel hit".
// Object ids in the incidence lists ("dd ids"): [0, nT5) T5, then pT5, then pT3.
#include "lst_launch.h"

namespace lst {

struct DRef {
  int type;              // 0 T5, 1 pT5, 2 pT3
  uint32_t idx;          // index inside its own collection
  int n_ot;              // 10 or 6
  const uint32_t *hits;  // sorted hit positions, layer order
  uint32_t pls;
  double score;
};

__device__ __forceinline__ DRef dd_ref(const SlotDev &s, uint32_t n5, uint32_t np5, uint32_t d) {
  DRef r;
  if (d < n5) {
    r.type = 0; r.idx = d; r.n_ot = 10; r.hits = s.t5_hits + 10 * (size_t)d; r.pls = 0xFFFFFFFFu; r.score = s.t5_chi2[d];
  } else if (d < n5 + np5) {
    const uint32_t i = d - n5;
    const uint2 po = s.pt5_po[i];
    r.type = 1; r.idx = i; r.n_ot = 10; r.hits = s.t5_hits + 10 * (size_t)po.y; r.pls = po.x; r.score = s.pt5_chi2[i];
  } else {
    const uint32_t i = d - n5 - np5;
    r.type = 2; r.idx = i; r.n_ot = 6; r.hits = s.pt3_hits + 6 * (size_t)i; r.pls = s.pt3_po[i].x; r.score = s.pt3_chi2[i];
  }
  return r;
}
__device__ __forceinline__ int dd_type(uint32_t n5, uint32_t np5, uint32_t d) { return d < n5 ? 0 : (d < n5 + np5 ? 1 : 2); }

// "b beats a": (score, hit coordinates in layer order, pLS index, original hit indices), reading 15.
// the tie-break of equal scores (rare: kept out of line so that its loads are not speculated)
__device__ __noinline__ bool dd_beats_tie(const SlotDev &s, const DRef &b, const DRef &a);
__device__ __forceinline__ bool dd_beats(const SlotDev &s, const DRef &b, const DRef &a) {
  if (b.score < a.score) return true;
  if (b.score > a.score) return false;
  return dd_beats_tie(s, b, a);
}
__device__ __noinline__ bool dd_beats_tie(const SlotDev &s, const DRef &b, const DRef &a) {
  const int n = a.n_ot < b.n_ot ? a.n_ot : b.n_ot;
  for (int k = 0; k < n; ++k) {
    const float4 pb = s.hit[b.hits[k]], pa = s.hit[a.hits[k]];
    if (pb.x < pa.x) return true;
    if (pb.x > pa.x) return false;
    if (pb.y < pa.y) return true;
    if (pb.y > pa.y) return false;
    if (pb.z < pa.z) return true;
    if (pb.z > pa.z) return false;
  }
  if (a.type != 0 && b.type != 0) {
    if (b.pls < a.pls) return true;
    if (b.pls > a.pls) return false;
  }
  for (int k = 0; k < n; ++k) {
    const uint32_t ob = s.hit_orig[b.hits[k]], oa = s.hit_orig[a.hits[k]];
    if (ob < oa) return true;
    if (ob > oa) return false;
  }
  return false;
}

__device__ __forceinline__ int dd_shared(const uint32_t *ha, int na, const uint32_t *hb, int nb) {
  int n = 0;
  for (int j = 0; j < nb; ++j) {
    const uint32_t v = hb[j];
#pragma unroll
    for (int i = 0; i < 10; ++i) n += (i < na && ha[i] == v);
  }
  return n;
}

// The pixel-seed lookups (eta bins, seeds close to a seed, the hash set of the pixel-hit ids) are built
// by the seed kernels of k_pix.cu; here they are only read.
__device__ __forceinline__ void pid_mark(const SlotDev &s, uint8_t *flag, uint32_t p) {
  const uint4 sl = reinterpret_cast<const uint4 *>(s.pls_slot)[p];
  flag[sl.x] = 1; flag[sl.y] = 1; flag[sl.z] = 1; flag[sl.w] = 1;
}
__device__ __forceinline__ bool pid_any(const SlotDev &s, uint32_t p, bool with3) {
  const uint4 sl = reinterpret_cast<const uint4 *>(s.pls_slot)[p];
  uint32_t v = s.pid_has5[sl.x] | s.pid_has5[sl.y] | s.pid_has5[sl.z] | s.pid_has5[sl.w];
  if (with3) v |= s.pid_has3[sl.x] | s.pid_has3[sl.y] | s.pid_has3[sl.z] | s.pid_has3[sl.w];
  return v != 0;
}

// ------------------------------------------------------------------ hit -> objects incidence
__device__ __forceinline__ void md_hits2(const SlotDev &s, uint32_t md, uint32_t *out) {
  const uint2 h = s.md_hit[md];
  out[0] = h.x; out[1] = h.y;
}
// thread per dd object: gather its hit positions (T5 and pT3 store them) and count the incidences
__global__ void __launch_bounds__(256) k_dd_count(const __grid_constant__ Batch B, const __grid_constant__ Params g) {
  pdl_enter();
  LST_SLOT(B);
  const Header *hdr = s.hdr;
  {   // one warp per seed: the seeds close to it in eta-phi (S1, S3)
    const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t a = warp; a < hdr->n_seeds; a += nwarp) pls_adjacent(s, g, a);
  }
  const uint32_t n5 = hdr->n_obj[3], np5 = hdr->n_obj[5], n_dd = n5 + np5 + hdr->n_obj[4];
  for (uint32_t d = blockIdx.x * blockDim.x + threadIdx.x; d < n_dd; d += gridDim.x * blockDim.x) {
    uint32_t h[10];
    int n;
    if (d < n5 + np5) {
      const uint32_t t = d < n5 ? d : s.pt5_po[d - n5].y;
#pragma unroll
      for (int q = 0; q < 5; ++q) md_hits2(s, s.t5_md[5 * (size_t)t + q], h + 2 * q);
      n = 10;
      if (d < n5)
#pragma unroll
        for (int q = 0; q < 10; ++q) s.t5_hits[10 * (size_t)d + q] = h[q];
    } else {
      const uint32_t i = d - n5 - np5;
      const uint4 m = s.t3_md[s.pt3_po[i].y];
      md_hits2(s, m.x, h); md_hits2(s, m.y, h + 2); md_hits2(s, m.z, h + 4);
      n = 6;
#pragma unroll
      for (int q = 0; q < 6; ++q) s.pt3_hits[6 * (size_t)i + q] = h[q];
    }
    const uint32_t ty = (uint32_t)dd_type(n5, np5, d);
    for (int q = 0; q < n; ++q) atomicAdd(&s.inc_cnt[3 * h[q] + ty], 1u);
  }
}
__device__ __forceinline__ void pls_best_body(const SlotDev &s, uint32_t n5, uint32_t np5, uint32_t np3);
__global__ void __launch_bounds__(256) k_dd_scatter(const __grid_constant__ Batch B) {
  pdl_enter();
  LST_SLOT(B);
  const Header *hdr = s.hdr;
  const uint32_t n5 = hdr->n_obj[3], np5 = hdr->n_obj[5], np3 = hdr->n_obj[4], n_dd = n5 + np5 + np3;
  for (uint32_t d = blockIdx.x * blockDim.x + threadIdx.x; d < n_dd; d += gridDim.x * blockDim.x) {
    const DRef r = dd_ref(s, n5, np5, d);
    // the ten (six) rows are independent: all loads, then all atomics, then all stores in flight together
    uint32_t row[10], pos[10];
#pragma unroll
    for (int q = 0; q < 10; ++q) row[q] = q < r.n_ot ? 3 * r.hits[q] + (uint32_t)r.type : 0u;
#pragma unroll
    for (int q = 0; q < 10; ++q) pos[q] = q < r.n_ot ? s.inc_off[row[q]] : 0u;
#pragma unroll
    for (int q = 0; q < 10; ++q) if (q < r.n_ot) pos[q] += atomicAdd(&s.inc_cur[row[q]], 1u);
#pragma unroll
    for (int q = 0; q < 10; ++q) if (q < r.n_ot) s.inc_ent[pos[q]] = d;
  }
  pls_best_body(s, n5, np5, np3);
}

// ------------------------------------------------------------------ S0, same-seed rule
// "a is removed iff some b of the same pixel seed beats a" and "beats" is a strict total order, so
// of a seed's pT5 (pT3) exactly the minimum survives this rule.  One thread per object, two passes:
// the seed's minimum score by atomicMin on the bit pattern of the (non-negative) double, then the
// objects AT that score settle the tie order by compare-and-swap (anchors are lower hits, so T3 /
// T5 that differ only in upper hits tie exactly; the tie sets at the minimum are small).
// (the minimum is taken by the fill kernel of the pixel joins, k_t3t5.cu; the tie order here)
__device__ __forceinline__ void pls_best_body(const SlotDev &s, uint32_t n5, uint32_t np5, uint32_t np3) {
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < np5 + np3; j += gridDim.x * blockDim.x) {
    const bool is5 = j < np5;
    const uint32_t i = is5 ? j : j - np5;
    const uint32_t p = (is5 ? s.pt5_po : s.pt3_po)[i].x;
    const double sc = (is5 ? s.pt5_chi2 : s.pt3_chi2)[i];
    if ((unsigned long long)__double_as_longlong(sc) != (is5 ? s.pls_min5 : s.pls_min3)[p]) continue;
    uint32_t *best = (is5 ? s.pls_best5 : s.pls_best3) + p;
    const uint32_t dbase = is5 ? n5 : n5 + np5;
    const DRef me = dd_ref(s, n5, np5, dbase + i);
    uint32_t cur = *(volatile uint32_t *)best;
    while (cur == 0xFFFFFFFFu || dd_beats_tie(s, me, dd_ref(s, n5, np5, dbase + cur))) {
      const uint32_t old = atomicCAS(best, cur, i);
      if (old == cur) break;
      cur = old;
    }
  }
}

// ------------------------------------------------------------------ S0: inside one collection
// EIGHT LANES per object A, four objects per warp (most objects are beaten by one of the first few
// entries they look at, so the per-object set-up dominates; it is shared by four objects here).
// An object sharing >= min_shared of A's n_ot hits contains at least one of any n_ot - min_shared
// + 1 of them, so only the n_ot - min_shared + 1 shortest incidence lists (of A's own type) are
// searched; the lists are flattened into one index space that the 8 lanes stride.  Per entry B the
// cheap test comes first (score(B) <= score(A)); the shared-hit count is exact and costs one
// shared-memory lookup per hit of B: A's hits sit in a 128-slot table per group (slot = hit & 127;
// an A whose hits collide in the table counts with the 10 x 10 comparison instead).
constexpr int kS0Slots = 128;
constexpr uint32_t kNoHit = 0xFFFFFFFFu;
constexpr uint32_t kS0Light = 64;   // entries an 8-lane group looks at before it hands a longer object to k_s0_heavy
//
// pass > 0 (lst_config.s0_fixpoint_passes): a pass of the fix-point iteration of the T5 collection.  The
// non-greedy rule (pass 0) keeps L1 = {no better duplicate at all}; pass p keeps {no better duplicate
// among the objects kept by pass p - 1}.  The passes alternate between subsets (even p) and supersets
// (odd p) of the greedy fix-point "kept iff no KEPT better duplicate" and meet it after a few steps; the
// flags of pass p - 1 are read from one of two buffers (t5_keep, t5_keep2), those of pass p go to the other.
__global__ void __launch_bounds__(128) k_s0(const __grid_constant__ Batch B, const __grid_constant__ Params g, int pass,
                                            int last_pass) {
  __shared__ uint32_t sh_pre[16][12], sh_beg[16][12];
  __shared__ uint32_t sh_tab[16][kS0Slots];
  pdl_enter();
  LST_SLOT(B);
  Header *hdr = s.hdr;
  const uint32_t n5 = hdr->n_obj[3], np5 = hdr->n_obj[5], n_dd = n5 + np5 + hdr->n_obj[4];
  const uint8_t *alive = pass == 0 ? nullptr : ((pass & 1) ? s.t5_keep : s.t5_keep2);     // flags of the previous pass
  uint8_t *t5_out = (pass & 1) ? s.t5_keep2 : s.t5_keep;
  const int lane = threadIdx.x & 31, gl = lane & 7, gbase = lane & ~7, gid = threadIdx.x >> 3;
  const uint32_t gmask = 0xFFu << gbase;
  const uint32_t group = (blockIdx.x * blockDim.x + threadIdx.x) >> 3, ngroup = (gridDim.x * blockDim.x) >> 3;
  uint32_t *pre = sh_pre[gid], *beg = sh_beg[gid], *tab = sh_tab[gid];
  for (int k = gl; k < kS0Slots; k += 8) tab[k] = kNoHit;
  __syncwarp();
  // Same-seed rule first: of a seed's pT5 (pT3) only its best can survive, whatever the shared-hit search
  // says, so the others are flagged here and the search below runs on the T5 and on the seeds' best
  // objects only (work index: [0, n5) T5, then per seed its best pT5, then per seed its best pT3).
  const uint32_t n_seeds = hdr->n_seeds;
  if (g.s0_enabled && pass == 0) {
    const uint32_t np3 = hdr->n_obj[4];
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < np5 + np3; j += gridDim.x * blockDim.x) {
      if (j < np5) { if (s.pls_best5[s.pt5_po[j].x] != j) s.pt5_keep[j] = 0; }
      else { const uint32_t i = j - np5; if (s.pls_best3[s.pt3_po[i].x] != i) s.pt3_keep[i] = 0; }
    }
  }
  const uint32_t n_work = pass ? n5 : (g.s0_enabled ? n5 + 2u * n_seeds : n_dd);
  for (uint32_t wk = group;; wk += ngroup) {
    if (!__any_sync(0xffffffffu, wk < n_work)) break;
    uint32_t d = wk;
    bool valid = wk < n_work;
    if (valid && g.s0_enabled && wk >= n5) {
      const uint32_t q = wk - n5, best = q < n_seeds ? s.pls_best5[q] : s.pls_best3[q - n_seeds];
      valid = best != 0xFFFFFFFFu;
      d = (q < n_seeds ? n5 : n5 + np5) + best;
    }
    DRef A;
    A.type = 0; A.idx = 0; A.n_ot = 0; A.hits = nullptr; A.pls = kNoHit; A.score = 0.0;
    if (valid) A = dd_ref(s, n5, np5, d);
    // lane gl owns hits gl and gl + 8 of A
    const uint32_t h0 = gl < A.n_ot ? A.hits[gl] : kNoHit, h1 = gl + 8 < A.n_ot ? A.hits[gl + 8] : kNoHit;
    bool beaten = false, defer = false;
    if (g.s0_enabled) {
      const int min_shared = A.type == 0 ? g.dup_t5 : (A.type == 1 ? g.dup_pt5 : g.dup_pt3);
      const int k0 = min_shared - 1, nl = A.n_ot > k0 ? A.n_ot - k0 : 0;   // number of lists searched
      // table of A's hits; a collision (two hits of A in one slot) -> exact comparison path
      const uint32_t slot0 = h0 & (kS0Slots - 1), slot1 = h1 & (kS0Slots - 1);
      if (h0 != kNoHit) tab[slot0] = h0;
      __syncwarp();
      if (h1 != kNoHit) tab[slot1] = h1;
      __syncwarp();
      const bool bad = (h0 != kNoHit && tab[slot0] != h0) || (h1 != kNoHit && tab[slot1] != h1);
      const bool collide = (__ballot_sync(0xffffffffu, bad) & gmask) != 0u;
      {
        // the nl SHORTEST of A's n_ot incidence lists are searched (any nl of them will do)
        uint32_t len0 = 0, b0 = 0, len1 = 0, b1 = 0;
        if (h0 != kNoHit) { const uint32_t row = 3 * h0 + (uint32_t)A.type; b0 = s.inc_off[row]; len0 = s.inc_off[row + 1] - b0; }
        if (h1 != kNoHit) { const uint32_t row = 3 * h1 + (uint32_t)A.type; b1 = s.inc_off[row]; len1 = s.inc_off[row + 1] - b1; }
        // rank by (length, hit position): keys are unique, missing hits sort last
        const uint32_t key0 = h0 != kNoHit ? ((len0 < (1u << 27) ? len0 : (1u << 27) - 1u) << 4) | (uint32_t)gl : kNoHit;
        const uint32_t key1 = h1 != kNoHit ? ((len1 < (1u << 27) ? len1 : (1u << 27) - 1u) << 4) | (uint32_t)(gl + 8) : kNoHit;
        int rank0 = 0, rank1 = 0;
#pragma unroll
        for (int j = 0; j < 10; ++j) {
          const uint32_t kj = j < 8 ? __shfl_sync(0xffffffffu, key0, gbase | j) : __shfl_sync(0xffffffffu, key1, gbase | (j - 8));
          rank0 += (int)(kj < key0); rank1 += (int)(kj < key1);
        }
        if (h0 != kNoHit && rank0 < nl) { beg[rank0] = b0; pre[rank0] = len0; }
        if (h1 != kNoHit && rank1 < nl) { beg[rank1] = b1; pre[rank1] = len1; }
        __syncwarp();
        if (gl == 0) {                                           // exclusive prefix of the <= 10 selected lengths
          uint32_t acc = 0;
          for (int q = 0; q < nl; ++q) { const uint32_t t = pre[q]; pre[q] = acc; acc += t; }
          pre[nl] = acc;
        }
        __syncwarp();
      }
      const uint32_t total = valid ? pre[nl] : 0u;
      const double *score_arr = A.type == 0 ? s.t5_chi2 : (A.type == 1 ? s.pt5_chi2 : s.pt3_chi2);
      const uint32_t dbase = A.type == 0 ? 0u : (A.type == 1 ? n5 : n5 + np5);
      int cur = 0;
      for (uint32_t base = 0;; base += 8) {
        if (!beaten && base >= kS0Light && base < total) defer = true;     // a long one: the whole-warp kernel takes it
        const bool active = !beaten && !defer && base < total;
        if (!__any_sync(0xffffffffu, active)) break;
        const uint32_t i = base + gl;
        bool hit = false;
        if (active && i < total) {
          while (i >= pre[cur + 1]) ++cur;
          const uint32_t b = s.inc_ent[beg[cur] + (i - pre[cur])];
          if (b != d && !(score_arr[b - dbase] > A.score) && (alive == nullptr || alive[b])) {
            int cnt;
            if (!collide) {
              const uint32_t *hb = A.type == 0 ? s.t5_hits + 10 * (size_t)b
                                 : (A.type == 1 ? s.t5_hits + 10 * (size_t)s.pt5_po[b - dbase].y
                                                : s.pt3_hits + 6 * (size_t)(b - dbase));
              const uint2 *hb2 = reinterpret_cast<const uint2 *>(hb);
              cnt = 0;
#pragma unroll
              for (int q = 0; q < 5; ++q) {
                if (2 * q < A.n_ot) {
                  const uint2 v = hb2[q];
                  cnt += (int)(tab[v.x & (kS0Slots - 1)] == v.x) + (int)(tab[v.y & (kS0Slots - 1)] == v.y);
                }
              }
            } else {
              uint32_t ha[10];
#pragma unroll
              for (int q = 0; q < 10; ++q) ha[q] = q < A.n_ot ? A.hits[q] : kNoHit;
              const DRef Bq = dd_ref(s, n5, np5, b);
              cnt = dd_shared(ha, A.n_ot, Bq.hits, Bq.n_ot);
            }
            if (cnt >= min_shared) hit = dd_beats(s, dd_ref(s, n5, np5, b), A);
          }
        }
        if ((__ballot_sync(0xffffffffu, hit) & gmask) != 0u) beaten = true;
      }
      // objects of the same pixel seed are duplicates of one another: only the seed's best survives
      if (valid && A.type != 0 && (A.type == 1 ? s.pls_best5 : s.pls_best3)[A.pls] != A.idx) beaten = true;
      __syncwarp();
      if (h0 != kNoHit) tab[slot0] = kNoHit;                     // leave the table empty for the next object
      if (h1 != kNoHit) tab[slot1] = kNoHit;
      __syncwarp();
    }
    if (valid && gl == 0 && defer && !beaten) s.tc_pos[atomicAdd(&hdr->n_heavy[pass], 1u)] = d;
    if (valid && gl == 0 && !(defer && !beaten)) {
      const bool keep = !beaten;
      if (A.type == 0) {
        t5_out[A.idx] = keep;
        if (last_pass && alive && (alive[A.idx] != 0) != keep) atomicAdd(&hdr->n_unsettled, 1u);
      }
      else if (A.type == 1) {
        s.pt5_keep[A.idx] = keep;
        if (keep) {
          s.pls_has5[A.pls] = 1;
          pid_mark(s, s.pid_has5, A.pls);
          for (int q = 0; q < 10; ++q) s.hit_used5[A.hits[q]] = 1;   // S1 / S2: "shares a hit with a surviving pT5"
        }
      }
      else s.pt3_keep[A.idx] = keep;
    }
  }
}

// The objects k_s0 deferred (not beaten by their first kS0Light entries and with longer lists: mostly
// the objects that survive): one BLOCK per object over the whole flattened list (a hit of a |eta| ~ 0
// seed's objects is shared by thousands of pT3: the longest lists set the duration, so they get 128
// lanes), objects handed out dynamically.  Warp 0 sets the object up, all warps stride the list.
__global__ void __launch_bounds__(128) k_s0_heavy(const __grid_constant__ Batch B, const __grid_constant__ Params g, int pass,
                                                  int last_pass) {
  __shared__ uint32_t pre[12], beg[12];
  __shared__ uint32_t tab[256];
  __shared__ uint32_t sh_hv, sh_collide;
  pdl_enter();
  LST_SLOT(B);
  const Header *hdr = s.hdr;
  const uint32_t n5 = hdr->n_obj[3], np5 = hdr->n_obj[5], n_heavy = hdr->n_heavy[pass];
  const uint8_t *alive = pass == 0 ? nullptr : ((pass & 1) ? s.t5_keep : s.t5_keep2);
  uint8_t *t5_out = (pass & 1) ? s.t5_keep2 : s.t5_keep;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  for (int k = threadIdx.x; k < 256; k += blockDim.x) tab[k] = 0xFFFFFFFFu;
  for (;;) {
    __syncthreads();                                            // the previous object is done with the shared arrays
    if (threadIdx.x == 0) sh_hv = atomicAdd(&s.hdr->heavy_next[pass], 1u);
    __syncthreads();
    const uint32_t hv = sh_hv;
    if (hv >= n_heavy) break;
    const uint32_t d = s.tc_pos[hv];
    const DRef A = dd_ref(s, n5, np5, d);
    const int min_shared = A.type == 0 ? g.dup_t5 : (A.type == 1 ? g.dup_pt5 : g.dup_pt3);
    const int k0 = min_shared - 1, nl = A.n_ot > k0 ? A.n_ot - k0 : 0;   // number of lists searched
    bool beaten = false;
    if (g.s0_enabled) {
      uint32_t slot = 0;
      if (wib == 0) {
        // lane q < n_ot owns hit q of A: table of A's hits; collisions (two hits of A in one slot) ->
        // exact comparison path
        const uint32_t my_hit = lane < A.n_ot ? A.hits[lane] : 0xFFFFFFFFu;
        slot = my_hit & (256 - 1);
        const uint32_t same = __match_any_sync(0xffffffffu, lane < A.n_ot ? slot : 0x10000u + lane);
        const bool collide = __any_sync(0xffffffffu, lane < A.n_ot && __popc(same) > 1);
        if (lane < A.n_ot) tab[slot] = my_hit;
        if (lane == 0) sh_collide = collide;
        // the nl SHORTEST of A's n_ot incidence lists are searched (any nl of them will do)
        uint32_t len = 0, b0 = 0;
        if (lane < A.n_ot) {
          const uint32_t row = 3 * my_hit + (uint32_t)A.type;
          b0 = s.inc_off[row]; len = s.inc_off[row + 1] - b0;
        }
        // rank of this lane's list by (length, lane): keys are unique, lanes >= n_ot sort last
        const uint32_t mykey = lane < A.n_ot ? ((len < (1u << 27) ? len : (1u << 27) - 1u) << 4) | (uint32_t)lane : 0xFFFFFFFFu;
        int rank = 0;
#pragma unroll
        for (int j = 0; j < 10; ++j) rank += (int)(__shfl_sync(0xffffffffu, mykey, j) < mykey);
        if (lane < A.n_ot && rank < nl) { beg[rank] = b0; pre[rank] = len; }
        __syncwarp();
        const uint32_t l2 = lane < nl ? pre[lane] : 0u;
        uint32_t tot;
        const uint32_t ex = warp_excl_scan(l2, &tot);
        __syncwarp();
        if (lane < 11) pre[lane] = ex;                          // lanes >= nl: pre = total
      }
      __syncthreads();
      const bool collide = sh_collide != 0u;
      const uint32_t total = pre[nl < 10 ? nl : 10];
      const double *score_arr = A.type == 0 ? s.t5_chi2 : (A.type == 1 ? s.pt5_chi2 : s.pt3_chi2);
      const uint32_t dbase = A.type == 0 ? 0u : (A.type == 1 ? n5 : n5 + np5);
      int cur = 0;
      for (uint32_t base = 0; base < total && !beaten; base += blockDim.x) {
        const uint32_t i = base + threadIdx.x;
        bool hit = false;
        if (i < total) {
          while (i >= pre[cur + 1]) ++cur;
          const uint32_t b = s.inc_ent[beg[cur] + (i - pre[cur])];
          if (b != d && !(score_arr[b - dbase] > A.score) && (alive == nullptr || alive[b])) {
            int cnt;
            if (!collide) {
              const uint32_t *hb = A.type == 0 ? s.t5_hits + 10 * (size_t)b
                                 : (A.type == 1 ? s.t5_hits + 10 * (size_t)s.pt5_po[b - dbase].y
                                                : s.pt3_hits + 6 * (size_t)(b - dbase));
              const uint2 *hb2 = reinterpret_cast<const uint2 *>(hb);
              cnt = 0;
#pragma unroll
              for (int q = 0; q < 5; ++q) {
                if (2 * q < A.n_ot) {
                  const uint2 v = hb2[q];
                  cnt += (int)(tab[v.x & (256 - 1)] == v.x) + (int)(tab[v.y & (256 - 1)] == v.y);
                }
              }
            } else {
              uint32_t ha[10];
#pragma unroll
              for (int q = 0; q < 10; ++q) ha[q] = q < A.n_ot ? A.hits[q] : 0xFFFFFFFFu;
              const DRef Bq = dd_ref(s, n5, np5, b);
              cnt = dd_shared(ha, A.n_ot, Bq.hits, Bq.n_ot);
            }
            if (cnt >= min_shared) hit = dd_beats(s, dd_ref(s, n5, np5, b), A);
          }
        }
        beaten = __syncthreads_or(hit) != 0;
      }
      __syncthreads();
      if (wib == 0 && lane < A.n_ot) tab[slot] = 0xFFFFFFFFu;     // leave the table empty for the next object
      // objects of the same pixel seed are duplicates of one another: only the seed's best survives
      if (!beaten && A.type != 0 && (A.type == 1 ? s.pls_best5 : s.pls_best3)[A.pls] != A.idx) beaten = true;
    }
    if (threadIdx.x == 0) {
      const bool keep = !beaten;
      if (A.type == 0) {
        t5_out[A.idx] = keep;
        if (last_pass && alive && (alive[A.idx] != 0) != keep) atomicAdd(&s.hdr->n_unsettled, 1u);
      }
      else if (A.type == 1) {
        s.pt5_keep[A.idx] = keep;
        if (keep) {
          s.pls_has5[A.pls] = 1;
          pid_mark(s, s.pid_has5, A.pls);
          for (int q = 0; q < 10; ++q) s.hit_used5[A.hits[q]] = 1;   // S1 / S2: "shares a hit with a surviving pT5"
        }
      }
      else s.pt3_keep[A.idx] = keep;
    }
  }
}

// ------------------------------------------------------------------ S1: pT3 against surviving pT5
__global__ void __launch_bounds__(128) k_s1(const __grid_constant__ Batch B) {
  pdl_enter();
  LST_SLOT(B);
  const Header *hdr = s.hdr;
  const uint32_t np3 = hdr->n_obj[4];
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < np3; i += gridDim.x * blockDim.x) {
    if (!s.pt3_keep[i]) continue;
    const uint32_t p = s.pt3_po[i].x;
    bool dup = s.pls_has5[p] || pid_any(s, p, false);
    const uint32_t na = s.pls_adj_cnt[p];
    for (uint32_t k = 0; k < na && !dup; ++k) dup = s.pls_has5[s.pls_adj[(size_t)p * kAdjCap + k]];
    uint32_t h[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) h[q] = s.pt3_hits[6 * (size_t)i + q];
#pragma unroll
    for (int q = 0; q < 6; ++q) dup |= (s.hit_used5[h[q]] != 0);
    if (dup) s.pt3_keep[i] = 0;
    else {
      s.pls_has3[p] = 1;
      pid_mark(s, s.pid_has3, p);
#pragma unroll
      for (int q = 0; q < 6; ++q) s.hit_used3[h[q]] = 1;
    }
  }
}

// ------------------------------------------------------------------ S2: T5 against surviving pT5 / pT3
// A warp takes 32 T5 at a time (lane = object: keep flag and the ten hit flags), then the objects
// still alive one by one, all lanes striding over the seeds of the object's eta bins (the loops over
// ~30 binned seeds with fp64 distance tests were the latency of the thread-per-object version).
__global__ void __launch_bounds__(128) k_s2(const __grid_constant__ Batch B, const __grid_constant__ Params g) {
  pdl_enter();
  LST_SLOT(B);
  const Header *hdr = s.hdr;
  const uint32_t n5 = hdr->n_obj[3];
  const int lane = threadIdx.x & 31;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
  for (uint32_t base = warp * 32; base < n5; base += nwarp * 32) {
    const uint32_t i = base + lane;
    bool alive = i < n5 && s.t5_keep[i] != 0;
    if (alive) {
      bool dup = false;
#pragma unroll
      for (int q = 0; q < 10; ++q) {
        const uint32_t h = s.t5_hits[10 * (size_t)i + q];
        dup |= (s.hit_used5[h] | s.hit_used3[h]) != 0;
      }
      if (dup) { s.t5_keep[i] = 0; alive = false; }
    }
    uint32_t todo = __ballot_sync(0xffffffffu, alive);
    while (todo) {
      const int src = __ffs(todo) - 1;
      todo &= todo - 1;
      const uint32_t o = base + src;
      const double2 ep = s.t5_etaphi[o];
      const int b0 = eta_bin(g, ep.x);
      const int lo = b0 > 0 ? b0 - 1 : 0, hi = b0 + 1 < g.eta_nbins ? b0 + 1 : g.eta_nbins - 1;
      const uint32_t e0 = s.pls_bin_off[lo], e1 = s.pls_bin_off[hi + 1];
      bool dup = false;
      uint32_t near_mask_any = 0;
      for (uint32_t eb = e0; eb < e1; eb += 32) {
        const uint32_t e = eb + lane;
        bool close = false, used = false;
        if (e < e1) {
          const uint32_t p = s.pls_bin_ent[e];
          close = close_eta_phi(g, ep.x, ep.y, (double)s.seed_eta[p], (double)s.seed_phi[p]);
          used = close && (s.pls_has5[p] || s.pls_has3[p]);
        }
        dup |= __any_sync(0xffffffffu, used);
        near_mask_any |= __ballot_sync(0xffffffffu, close);
      }
      if (dup) { if (lane == 0) s.t5_keep[o] = 0; continue; }
      if (near_mask_any == 0u) continue;
      for (uint32_t eb = e0; eb < e1; eb += 32) {   // survivor: the seeds close to it are duplicates of it (S3)
        const uint32_t e = eb + lane;
        if (e < e1) {
          const uint32_t p = s.pls_bin_ent[e];
          if (close_eta_phi(g, ep.x, ep.y, (double)s.seed_eta[p], (double)s.seed_phi[p])) s.pls_near_t5[p] = 1;
        }
      }
    }
  }
}

// ------------------------------------------------------------------ S3 + keep flags in TC order
__device__ __forceinline__ bool pls_unused(const SlotDev &s, uint32_t p) {
  return s.pt5_pls_off[p + 1] == s.pt5_pls_off[p] && s.pt3_pls_off[p + 1] == s.pt3_pls_off[p];
}
// Block b owns the flags [b C, (b + 1) C), C = ceil(n_flag / gridDim.x); it also counts them, and the
// last block to finish scans the per-block counts: k_tc_fill (same grid) places a kept entry at its
// block's offset + its rank inside the block.
__global__ void __launch_bounds__(256) k_s3_flags(const __grid_constant__ Batch B) {
  __shared__ uint32_t sh[33];
  pdl_enter();
  LST_SLOT(B);
  Header *hdr = s.hdr;
  const uint32_t n5 = hdr->n_obj[3], np5 = hdr->n_obj[5], np3 = hdr->n_obj[4], n = np5 + np3 + n5 + hdr->n_seeds;
  const uint32_t C = (n + gridDim.x - 1) / gridDim.x;
  const uint32_t i0 = min(n, blockIdx.x * C), i1 = min(n, i0 + C);
  uint32_t mine = 0;
  for (uint32_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) {
    uint32_t f;
    if (i < np5) f = s.pt5_keep[i];
    else if (i < np5 + np3) f = s.pt3_keep[i - np5];
    else if (i < np5 + np3 + n5) f = s.t5_keep[i - np5 - np3];
    else {
      const uint32_t p = i - np5 - np3 - n5;
      bool keep = pls_unused(s, p) && !s.pls_near_t5[p] && !pid_any(s, p, true);
      const uint32_t na = s.pls_adj_cnt[p];
      for (uint32_t k = 0; k < na && keep; ++k) {
        const uint32_t b = s.pls_adj[(size_t)p * kAdjCap + k];
        if (s.pls_has5[b] || s.pls_has3[b]) keep = false;
        else if (b < p && pls_unused(s, b)) keep = false;
      }
      s.pls_keep[p] = keep;
      f = keep;
    }
    s.tc_flag[i] = f;
    mine += f != 0u;
  }
  uint32_t tot;
  block_excl_scan(mine, sh, &tot);
  if (threadIdx.x == 0) s.flag_blk[blockIdx.x] = tot;
  if (!last_block(&hdr->ticket[TK_FLAGS], gridDim.x)) return;
  const uint32_t total = lb_scan_parts(s.flag_blk, gridDim.x, sh);
  if (threadIdx.x == 0) hdr->n_obj[6] = total;
}

// ------------------------------------------------------------------ S4: TC = pT5, pT3, T5, pLS survivors
__global__ void __launch_bounds__(256) k_tc_fill(const __grid_constant__ Batch B) {
  __shared__ uint32_t sh[33];
  pdl_enter();
  LST_SLOT(B);
  const Header *hdr = s.hdr;
  const uint32_t n5 = hdr->n_obj[3], np5 = hdr->n_obj[5], np3 = hdr->n_obj[4], n = np5 + np3 + n5 + hdr->n_seeds;
  const uint32_t C = (n + gridDim.x - 1) / gridDim.x;
  const uint32_t i0 = min(n, blockIdx.x * C), i1 = min(n, i0 + C);
  uint32_t carry = s.flag_blk[blockIdx.x];
  for (uint32_t base = i0; base < i1; base += blockDim.x) {
    const uint32_t i = base + threadIdx.x;
    const bool keep = i < i1 && s.tc_flag[i] != 0u;
    uint32_t tot;
    const uint32_t pos = carry + block_excl_scan(keep ? 1u : 0u, sh, &tot);
    carry += tot;
    if (keep) {
      uint32_t type, obj, p = 0xFFFFFFFFu;
      if (i < np5) { type = 5; obj = i; p = s.pt5_po[obj].x; }
      else if (i < np5 + np3) { type = 4; obj = i - np5; p = s.pt3_po[obj].x; }
      else if (i < np5 + np3 + n5) { type = 3; obj = i - np5 - np3; }
      else { type = 6; obj = i - np5 - np3 - n5; p = obj; }
      s.tc_to[pos] = make_uint2(type, obj);
      if (type == 3) {
        const double2 ep = s.t5_etaphi[obj];
        s.tc_f[pos] = make_float4(ld_f(s, s.t5_pt, obj), (float)ep.x, (float)ep.y, 3.0f);
      } else {
        s.tc_f[pos] = make_float4(s.seed_pt[p], s.seed_eta[p], s.seed_phi[p], (float)type);
      }
    }
    __syncthreads();
  }
}

static inline int grid_of(uint32_t n, int threads, int max_blocks) {
  long b = ((long)n + threads - 1) / threads;
  return (int)(b < 1 ? 1 : (b > max_blocks ? max_blocks : b));
}

// The zeroed scratch (incidence counters, seed / hit / pixel-id flags) and the 0xFF-filled per-seed
// minima are set by the two memsets at the start of the chain (lst_api.cu).
void launch_dedup(const Ctx &c, const Batch &b, cudaStream_t st) {
  const SlotDev &s = b.s[0];
  const uint32_t cap_dd = s.cap_t5 + s.cap_pt5 + s.cap_pt3;
  launch_k(c, st, "k_dd_count", k_dd_count, dim3(grid_of(cap_dd, 256, c.n_sm * 8)), 256, 0, false, b, c.par);
  launch_scan(c, b, 0, st);
  launch_k(c, st, "k_dd_scatter", k_dd_scatter, dim3(grid_of(cap_dd, 256, c.n_sm * 8)), 256, 0, false, b);
  for (int pass = 0; pass <= c.fix_passes; ++pass) {      // pass 0: the non-greedy rule; further passes: T5 fix-point iteration
    const int last = pass == c.fix_passes;
    const uint32_t n_obj = pass ? s.cap_t5 : cap_dd;
    launch_k(c, st, pass ? "k_s0[fix]" : "k_s0", k_s0, dim3(grid_of(n_obj, 16, c.n_sm * 16)), 128, 0, false, b, c.par, pass, last);
    launch_k(c, st, pass ? "k_s0_heavy[fix]" : "k_s0_heavy", k_s0_heavy, dim3(grid_of(n_obj, 4, c.n_sm * 16)), 128, 0, false, b,
             c.par, pass, last);
  }
  launch_k(c, st, "k_s1", k_s1, dim3(grid_of(s.cap_pt3, 128, c.n_sm * 16)), 128, 0, false, b);
  launch_k(c, st, "k_s2", k_s2, dim3(grid_of(s.cap_t5, 128, c.n_sm * 8)), 128, 0, false, b, c.par);
  launch_k(c, st, "k_s3_flags", k_s3_flags, dim3(kFlagBlocks), 256, 0, false, b);
  launch_k(c, st, "k_tc_fill", k_tc_fill, dim3(kFlagBlocks), 256, 0, false, b);
}

}  // namespace lst
