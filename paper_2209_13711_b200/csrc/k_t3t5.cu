// k_t3t5.cu -- a3 triplets (Fig. 5, 8; reading C4) and a4 quintuplets (PAPER.md:73,
// Fig. 9; reading C5: radius match, middle triplet, weighted Kasa circle-fit chi2).
//
// Both are joins on a shared mini-doublet: a T3 is LS (1,2) + LS (2,3), a T5 is T3 (1,2,3) +
// T3 (3,4,5).  Left objects are the rows; the right list of a row is the contiguous range of
// objects whose first MD is the row's last MD (LS are grouped by inner MD, T3 by first MD).
// Groups are chunks of kRowChunk rows; a group's candidates are numbered row-major.
#include "lst_launch.h"

namespace lst {

struct RowTab {                       // right-list table of one group, in shared memory
  uint32_t start[kRowChunk];
  uint32_t cum[kRowChunk + 1];
  uint32_t hint[kItemWords];          // row of the item's candidates 0, 32, 64, ... (stage_hints)
};

// KIND 0 (T3) : rows are LS, right lists are LS ranges of the outer MD.
// KIND 1 (T5) : rows are T3, right lists are T3 ranges of the third MD.
// KIND 2 (pT5): rows are (seed, compatible start module) pairs (k_pix.cu), right lists are the T5
//               whose first MD lies in that module (T5 are ordered by first MD, MDs by module).
// KIND 3 (pT3): same with T3.
enum { J_T3 = 0, J_T5 = 1, J_PT5 = 2, J_PT3 = 3 };

template <int KIND> struct JoinTraits;
template <> struct JoinTraits<J_T3> {
  static constexpr const char *n_groups = "k_join_groups[T3]", *n_eval = "k_join_eval[T3]", *n_decide = "k_join_decide[T3]", *n_fill = "k_join_fill[T3]";
  static constexpr int stage = S_T3, rows_level = 1, out_level = 2; };
template <> struct JoinTraits<J_T5> {
  static constexpr const char *n_groups = "k_join_groups[T5]", *n_eval = "k_join_eval[T5]", *n_decide = "k_join_decide[T5]", *n_fill = "k_join_fill[T5]";
  static constexpr int stage = S_T5, rows_level = 2, out_level = 3; };
template <> struct JoinTraits<J_PT5> {
  static constexpr const char *n_groups = "k_join_groups[pT5]", *n_eval = "k_join_eval[pT5]", *n_decide = "k_join_decide[pT5]", *n_fill = "k_join_fill[pT5]";
  static constexpr int stage = S_PT5, rows_level = kPairLevel, out_level = 5; };
template <> struct JoinTraits<J_PT3> {
  static constexpr const char *n_groups = "k_join_groups[pT3]", *n_eval = "k_join_eval[pT3]", *n_decide = "k_join_decide[pT3]", *n_fill = "k_join_fill[pT3]";
  static constexpr int stage = S_PT3, rows_level = kPairLevel, out_level = 4; };

template <int KIND>
__device__ __forceinline__ void right_range(const SlotDev &s, uint32_t row, uint32_t *st, uint32_t *cnt) {
  if (KIND == J_T3) {
    const uint32_t mo = s.ls_md[row].y;
    *st = s.ls_md_off[mo];
    *cnt = s.ls_md_off[mo + 1] - *st;
  } else if (KIND == J_T5) {
    const uint32_t m3 = s.t3_md[row].z;
    *st = s.t3_md_off[m3];
    *cnt = s.t3_md_off[m3 + 1] - *st;
  } else {
    // objects whose first MD lies in the row's module AND inside the row's azimuthal window (the MD
    // range k_px_modules found: objects are grouped by first MD)
    const uint2 rng = s.px_rng[row];
    const uint32_t *off = KIND == J_PT5 ? s.t5_md_off : s.t3_md_off;
    *st = off[rng.x];
    *cnt = off[rng.y] - *st;
  }
}

// Groups kernel body: one WARP per group (kRowChunk rows), kJoinGroupWarps groups per (virtual) block.
// Per row: first right object and the number of the group's candidates before the row (row_start,
// row_cum: the pre-filter kernel stages them, the fill kernel derives the CSR from them).  Per group:
// its candidate count and work items; first item of every group = exclusive prefix inside the
// virtual block here, across virtual blocks in the last block to finish.
constexpr int kJoinGroupWarps = 4;
template <int KIND>
__device__ __forceinline__ void join_groups_body(const SlotDev &s, uint32_t *sh_items, unsigned long long *sh_cand, uint32_t *sh) {
  const int stage = JoinTraits<KIND>::stage;
  const StageBuf &st = s.st[stage];
  Header *hdr = s.hdr;
  const uint32_t n_rows = hdr->n_obj[JoinTraits<KIND>::rows_level];
  const uint32_t ng = (n_rows + kRowChunk - 1) / kRowChunk;
  const uint32_t nvb = (ng + kJoinGroupWarps - 1) / kJoinGroupWarps;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  for (uint32_t vb = blockIdx.x; vb < nvb; vb += gridDim.x) {
    const uint32_t gidx = vb * kJoinGroupWarps + wib;
    uint32_t sum = 0;
    if (gidx < ng) {
      const uint32_t r0 = gidx * kRowChunk, r1 = min(r0 + kRowChunk, n_rows);
      for (uint32_t rb = r0; rb < r1; rb += 32) {
        const uint32_t r = rb + lane;
        uint32_t a = 0, c = 0;
        if (r < r1) right_range<KIND>(s, r, &a, &c);
        uint32_t tot;
        const uint32_t e = warp_excl_scan(c, &tot);
        if (r < r1) { st.row_start[r] = a; st.row_cum[r] = sum + e; }
        sum += tot;
      }
      if (lane == 0) { st.gR[gidx] = 1; st.gW[gidx] = sum; }
    }
    if (lane == 0) { sh_items[wib] = items_of(1u, sum); sh_cand[wib] = sum; }
    __syncthreads();
    if (threadIdx.x == 0) {
      uint32_t acc = 0;
      unsigned long long cs = 0;
      for (int k = 0; k < kJoinGroupWarps; ++k) {
        const uint32_t g = vb * kJoinGroupWarps + k;
        if (g < ng) st.g_item0[g] = acc;
        acc += sh_items[k]; cs += sh_cand[k];
      }
      st.gblk[vb] = acc;
      if (cs) atomicAdd(&hdr->cand[stage], cs);
    }
    __syncthreads();
  }
  if (!last_block(&hdr->ticket[TK_GROUPS + stage], gridDim.x)) return;
  const uint32_t total = lb_scan_parts(st.gblk, nvb, sh);
  lb_add_block_prefix(st.g_item0, ng, st.gblk, kJoinGroupWarps);
  if (threadIdx.x == 0) {
    const bool overflow = total > st.cap_items || ng > st.cap_groups;
    st.g_item0[ng] = total;
    hdr->n_groups[stage] = ng;
    hdr->n_items[stage] = overflow ? 0u : total;
    if (overflow) atomicOr(&hdr->err, (uint32_t)ERR_CAP_ITEMS);
  }
}
template <int KIND>
__global__ void __launch_bounds__(32 * kJoinGroupWarps) k_join_groups(const __grid_constant__ Batch B) {
  __shared__ uint32_t sh_items[kJoinGroupWarps];
  __shared__ unsigned long long sh_cand[kJoinGroupWarps];
  __shared__ uint32_t sh[33];
  pdl_enter();
  LST_SLOT(B);
  join_groups_body<KIND>(s, sh_items, sh_cand, sh);
}
// pT5 (blockIdx.y = 0) and pT3 (1) in one launch
__global__ void __launch_bounds__(32 * kJoinGroupWarps) k_px_groups(const __grid_constant__ Batch B) {
  __shared__ uint32_t sh_items[kJoinGroupWarps];
  __shared__ unsigned long long sh_cand[kJoinGroupWarps];
  __shared__ uint32_t sh[33];
  pdl_enter();
  LST_SLOT(B);
  if (blockIdx.y == 0) join_groups_body<J_PT5>(s, sh_items, sh_cand, sh);
  else join_groups_body<J_PT3>(s, sh_items, sh_cand, sh);
}

// the row table of a group from what the groups kernel stored
__device__ __forceinline__ void stage_rows(RowTab &rt, const StageBuf &st, uint32_t r0, uint32_t n_rows, uint32_t W) {
  const int tid = threadIdx.x;   // kThreads == kRowChunk
  const bool have = r0 + tid < n_rows;
  rt.start[tid] = have ? st.row_start[r0 + tid] : 0u;
  rt.cum[tid] = have ? st.row_cum[r0 + tid] : W;
  if (tid == 0) rt.cum[kRowChunk] = W;
  __syncthreads();
}
// flat candidate -> (row in group, right object)
__device__ __forceinline__ void flat_to_pair(const RowTab &rt, uint32_t cf, int *row, uint32_t *right) {
  int lo = 0, hi = kRowChunk;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (rt.cum[mid] <= cf) lo = mid; else hi = mid;
  }
  *row = lo;
  *right = rt.start[lo] + (cf - rt.cum[lo]);
}

// Per item: the row of every 32nd candidate, so that a candidate finds its row by a short linear
// walk (rows are ~100 candidates wide) instead of a 7-step binary search.
__device__ __forceinline__ void stage_hints(RowTab &rt, uint32_t j0) {
  if (threadIdx.x < kItemWords) {
    const uint32_t cf = j0 + 32u * threadIdx.x;
    int row = 0;
    if (cf < rt.cum[kRowChunk]) { uint32_t b; flat_to_pair(rt, cf, &row, &b); }
    rt.hint[threadIdx.x] = (uint32_t)row;
  }
  __syncthreads();
}
// candidate c of the item (flat index cf = j0 + c < total) -> (row in group, right object)
__device__ __forceinline__ void item_to_pair(const RowTab &rt, uint32_t j0, int c, int *row, uint32_t *right) {
  const uint32_t cf = j0 + (uint32_t)c;
  int r = (int)rt.hint[c >> 5];
  while (rt.cum[r + 1] <= cf) ++r;
  *row = r;
  *right = rt.start[r] + (cf - rt.cum[r]);
}

__device__ __forceinline__ Pt md_point(const SlotDev &s, uint32_t md) {
  const float4 p = s.md_pos[md];
  return make_pt(p.x, p.y, p.z, (int)(s.md_mod[md] & 3u));
}

// ------------------------------------------------------------------ evaluation of one candidate
__device__ __forceinline__ bool t3_candidate(const SlotDev &s, const Params &g, uint32_t a, uint32_t b, T3Out *o,
                                             uint4 *mds) {
  const uint2 la = s.ls_md[a], lb = s.ls_md[b];
  const Pt P1 = md_point(s, la.x), P2 = md_point(s, la.y), P3 = md_point(s, lb.y);
  if (mds) *mds = make_uint4(la.x, la.y, lb.y, 0u);
  return t3_eval_d(g, P1, P2, P3, o);
}
__device__ __forceinline__ bool t5_candidate(const SlotDev &s, const Params &g, uint32_t a, uint32_t b, T5Out *o,
                                             uint32_t *mds, double2 *ka, double2 *kb) {
  const double2 k3a = s.t3_kd[a], k3b = s.t3_kd[b];
  if (ka) { *ka = k3a; *kb = k3b; }
  if (!o && !le(fabs(k3a.x - k3b.x), g.ns * (k3a.y + k3b.y))) return false;   // early T5-1
  const uint4 ta = s.t3_md[a], tb = s.t3_md[b];
  const uint32_t m[5] = {ta.x, ta.y, ta.z, tb.y, tb.z};
  Pt P[5];
#pragma unroll
  for (int k = 0; k < 5; ++k) { P[k] = md_point(s, m[k]); if (mds) mds[k] = m[k]; }
  return t5_eval_d(g, P, k3a.x, k3a.y, k3b.x, k3b.y, o);
}

// pT5 / pT3 candidate: pixel seed against OT object `obj` (reading C6).  The fp32 pre-filter tests
// the first and the last anchor, loosened by kPreSlack plus absolute slacks far above the fp32 error
// (1e-5 rad on a >= 4e-3 rad window, 2e-3 cm on a >= 0.2 cm window); it never rejects on NaN.
// sp = {kappa_p, sinh eta, phi, z0} of the seed, computed once per row (stage_seeds).
// one anchor (MD m) against the seed parameters sp
__device__ __forceinline__ bool px_anchor_f(const SlotDev &s, const Params &g, float4 sp, uint32_t m) {
  const float4 h = s.md_pos[m];
  const int cat = (int)(s.md_mod[m] & 3u);
  const float kp = sp.x, sh = sp.y;
  float al;
  if (cat < 2) {
    const float kr = kp * h.w;
    al = fabsf(kr) <= 1e-4f ? h.w : __fdividef(asinf(fminf(1.0f, fmaxf(-1.0f, kr))), kp);
  } else {
    al = __fdividef(h.z - sp.w, sh);
  }
  const float d = s.md_phi[m] - (sp.z + kp * al);
  const float dph = d - 6.2831853071795864769f * rintf(d * 0.15915494309189533577f);
  const float sgp = (float)g.seed_sig_phi + (float)g.seed_sig_pt * fabsf(kp) * al + __fdividef(g.f_sig_t[cat], h.w);
  if (fabsf(dph) > g.f_ns * sgp * kPreSlack + 1e-5f) return false;
  float dzt, szt;
  if (cat < 2) {
    dzt = h.z - (sp.w + sh * al);
    szt = (float)g.seed_sig_z + g.f_sig_z[cat];
  } else {
    const float ka = kp * al;
    dzt = h.w - (fabsf(ka) <= 1e-4f ? al : __fdividef(sinf(ka), kp));
    szt = __fdividef((float)g.seed_sig_z, fabsf(sh)) + g.f_sig_r[cat];
  }
  if (fabsf(dzt) > g.f_ns * szt * kPreSlack + 2e-3f) return false;
  return true;
}
// first and last anchor of the object (the last one has the longest lever arm: together they leave
// the fp64 kernel little more than the accepted pairs)
template <int KIND>
__device__ __forceinline__ bool px_pre_f(const SlotDev &s, const Params &g, float4 sp, uint32_t obj) {
  uint32_t m0, m1;
  if (KIND == J_PT5) { m0 = s.t5_md[5 * (size_t)obj]; m1 = s.t5_md[5 * (size_t)obj + 4]; }
  else { const uint4 t = s.t3_md[obj]; m0 = t.x; m1 = t.z; }
  return px_anchor_f(s, g, sp, m0) && px_anchor_f(s, g, sp, m1);
}

// fp64 decision (and chi2_pix) of one (seed, object) pair.
template <int KIND>
__device__ __forceinline__ bool px_candidate(const GeoDev &geo, const SlotDev &s, const Params &g, uint32_t p,
                                             uint32_t obj, double *chi2) {
  constexpr int N = KIND == J_PT5 ? 5 : 3;
  uint32_t m[5];
  if (KIND == J_PT5) {
#pragma unroll
    for (int k = 0; k < 5; ++k) m[k] = s.t5_md[5 * (size_t)obj + k];
  } else {
    const uint4 t = s.t3_md[obj];
    m[0] = t.x; m[1] = t.y; m[2] = t.z;
  }
  Seed sd;
  sd.pt = (double)s.seed_pt[p]; sd.eta = (double)s.seed_eta[p]; sd.phi = (double)s.seed_phi[p];
  sd.z0 = (double)s.seed_z0[p]; sd.q = s.seed_q[p];
  Pt P[N];
#pragma unroll
  for (int k = 0; k < N; ++k) P[k] = md_point(s, m[k]);
  double c2 = 0.0;
  const bool ok = px_eval_d(g, sd, P, N, (int)geo.layer[s.md_mod[m[0]] >> 2], &c2);
  if (chi2) *chi2 = c2;
  return ok;
}

// What a row contributes to every one of its candidates, staged once per group in shared memory
// (T3: the anchors of the row LS; T5: kappa3 of the row T3 and the anchors of its MDs 2, 3; pixel: the
// seed parameters {kappa_p, sinh eta, phi, z0} and the seed index).
struct RowData {
  float4 ra[kRowChunk], rb[kRowChunk];
  double2 rk[kRowChunk];
  uint32_t rc[kRowChunk];            // categories (ca | cb << 2), or the seed index
};
template <int KIND>
__device__ __forceinline__ void stage_rowdata(RowData &rd, const SlotDev &s, const Params &g, uint32_t r0, uint32_t n_rows) {
  const int tid = threadIdx.x;   // kThreads == kRowChunk
  const uint32_t row = r0 + tid;
  if (row >= n_rows) return;
  if (KIND == J_T3) {
    const uint2 la = s.ls_md[row];
    rd.ra[tid] = s.md_pos[la.x]; rd.rb[tid] = s.md_pos[la.y];
    rd.rc[tid] = (s.md_mod[la.x] & 3u) | ((s.md_mod[la.y] & 3u) << 2);
  } else if (KIND == J_T5) {
    const uint4 ta = s.t3_md[row];
    rd.rk[tid] = s.t3_kd[row];
    rd.ra[tid] = s.md_pos[ta.y]; rd.rb[tid] = s.md_pos[ta.z];
    rd.rc[tid] = (s.md_mod[ta.y] & 3u) | ((s.md_mod[ta.z] & 3u) << 2);
  } else {
    const uint32_t p = s.px_pair[row].x;
    rd.ra[tid] = make_float4(-(float)s.seed_q[p] * (float)g.kB / (2.0f * s.seed_pt[p]), sinhf(s.seed_eta[p]), s.seed_phi[p], s.seed_z0[p]);
    rd.rc[tid] = p;
  }
}

// Phase 1 of a join candidate: a cheap necessary condition evaluated on every candidate (T3: the
// fp32 pre-filter t3_pre_f; T5: the radius match T5-1 on the stored kappa3, then the middle triplet
// through t3_pre_f; pixel: the fp32 first / last anchor pre-filter).  *ab = the pair handed to the
// decide kernel.  (Splitting t3_pre_f into a cheap and an expensive part joined by a warp queue was
// measured and lost: the selective cut is T3-2, the expensive one.)
template <int KIND>
__device__ __forceinline__ bool join_phase1(const SlotDev &s, const Params &g, uint32_t row, uint32_t b,
                                            const RowData &rd, int lrow, uint2 *ab) {
  *ab = make_uint2(row, b);
  if (KIND == J_T3) {
    const uint32_t m3 = s.ls_md[b].y;
    const float4 p1 = rd.ra[lrow], p2 = rd.rb[lrow], p3 = s.md_pos[m3];
    const uint32_t cc = rd.rc[lrow];
    return t3_pre_f(g, p1.x, p1.y, p1.z, p1.w, (int)(cc & 3u), p2.x, p2.y, p2.z, p2.w, (int)(cc >> 2), p3.x, p3.y, p3.z, p3.w,
                    (int)(s.md_mod[m3] & 3u));
  }
  if (KIND == J_T5) {
    const double2 k3a = rd.rk[lrow], k3b = s.t3_kd[b];
    if (!le(fabs(k3a.x - k3b.x), g.ns * (k3a.y + k3b.y))) return false;          // T5-1 (exact, fp64)
    // T5-2: the middle triplet (MD 2, 3, 4) through the fp32 triplet pre-filter
    const uint32_t m4 = s.t3_md[b].y;
    const float4 p2 = rd.ra[lrow], p3 = rd.rb[lrow], p4 = s.md_pos[m4];
    const uint32_t cc = rd.rc[lrow];
    return t3_pre_f(g, p2.x, p2.y, p2.z, p2.w, (int)(cc & 3u), p3.x, p3.y, p3.z, p3.w, (int)(cc >> 2), p4.x, p4.y, p4.z, p4.w,
                    (int)(s.md_mod[m4] & 3u));
  }
  ab->x = rd.rc[lrow];          // the seed
  return px_pre_f<KIND>(s, g, rd.ra[lrow], b);
}
// Pre-filter kernel: every candidate of every group through phase 1; survivors go to the stage's
// candidate list.  A block takes a group (the pixel stages: a quarter of one, their candidate loops are
// latency bound and the groups few), stages its row table once and walks its work items (tiles of
// kItemCand candidates) with one barrier-free candidate loop each.
struct JoinSh {
  RowTab rt;
  RowData rd;
  ClStageT<64> cl_mem[kThreads / 32];
};
template <int KIND>
__device__ __forceinline__ void join_eval_body(const SlotDev &s, const Params &g, JoinSh &m) {
  ClBufT<64> cl;
  cl.init(&m.cl_mem[threadIdx.x >> 5]);
  const int stage = JoinTraits<KIND>::stage;
  const StageBuf &st = s.st[stage];
  const bool live = s.hdr->n_items[stage] != 0;            // 0: nothing to do, or the work list overflowed
  const uint32_t n_groups = live ? s.hdr->n_groups[stage] : 0u;
  const uint32_t n_rows = s.hdr->n_obj[JoinTraits<KIND>::rows_level];
  const int tid = threadIdx.x;
  constexpr uint32_t kSplit = (KIND == J_PT5 || KIND == J_PT3) ? 4u : 1u;
  constexpr int kPart = kItemCand / (int)kSplit;
  for (uint32_t v = blockIdx.x; v < n_groups * kSplit; v += gridDim.x) {
    const uint32_t grp = v / kSplit, part = v % kSplit;
    const uint32_t W = st.gW[grp];
    if (W == 0 || (part != 0 && W <= part * (uint32_t)kPart)) continue;   // uniform per block
    const uint32_t r0 = grp * kRowChunk, it0 = st.g_item0[grp];
    stage_rowdata<KIND>(m.rd, s, g, r0, n_rows);
    stage_rows(m.rt, st, r0, n_rows, W);
    for (uint32_t j0 = 0; j0 < W; j0 += kItemCand) {
      const uint32_t it = it0 + j0 / kItemCand;
      const int njt = (int)min((uint32_t)kItemCand, W - j0);
      if (part == 0 && tid < kItemWords) st.mask[(size_t)it * kItemWords + tid] = 0;   // the decide kernel ORs the pass bits in
      if ((int)(part * kPart) >= njt) continue;
      stage_hints(m.rt, j0);
      const uint32_t key0 = it * (uint32_t)kItemCand;
      const int nj = min(njt, (int)((part + 1) * kPart));
      for (int base = (int)(part * kPart); base < nj; base += kThreads) {
        const int c = base + tid;
        bool keep = false;
        uint2 ab = make_uint2(0u, 0u);
        if (c < nj) {
          int row; uint32_t b;
          item_to_pair(m.rt, j0, c, &row, &b);
          keep = join_phase1<KIND>(s, g, r0 + row, b, m.rd, row, &ab);
        }
        cl.push(s.hdr, st, stage, keep, key0 + (uint32_t)c, ab);
      }
      __syncthreads();                                       // the hints are rewritten by the next tile
    }
    __syncthreads();
  }
  cl.flush_all(s.hdr, st, stage);
}
template <int KIND>
__global__ void __launch_bounds__(kThreads, 10) k_join_eval(const __grid_constant__ Batch B, const __grid_constant__ Params g) {
  __shared__ JoinSh m;
  pdl_enter();
  LST_SLOT(B);
  join_eval_body<KIND>(s, g, m);
}
__global__ void __launch_bounds__(kThreads, 10) k_px_eval(const __grid_constant__ Batch B, const __grid_constant__ Params g) {
  __shared__ JoinSh m;
  pdl_enter();
  LST_SLOT(B);
  if (blockIdx.y == 0) join_eval_body<J_PT5>(s, g, m);
  else join_eval_body<J_PT3>(s, g, m);
}

// Decide kernel: the fp64 decision of the listed candidates, one thread each (dense warps, no
// staging); an accepted candidate sets its pass bit and writes its results to the stage's pool.
template <int KIND>
__device__ __forceinline__ void join_decide_body(const GeoDev &geo, const SlotDev &s, const Params &g) {
  const int stage = JoinTraits<KIND>::stage;
  const StageBuf &st = s.st[stage];
  Header *hdr = s.hdr;
  const uint32_t n = min(hdr->cl_used[stage], st.cap_cl);
  const uint32_t nround = (n + 31u) & ~31u;
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < nround; j += gridDim.x * blockDim.x) {
    const bool live = j < n;
    const uint32_t key = live ? st.cl_key[j] : 0u;
    const uint2 ab = live ? st.cl_ab[j] : make_uint2(0u, 0u);
    bool pass = false;
    if (KIND == J_T3) {
      T3Out o;
      if (live) pass = t3_candidate(s, g, ab.x, ab.y, &o, nullptr);
      if (pass) {
        st.p_d2[j] = make_double2(o.kappa3, o.sigk3);
        st.p_f4[j] = make_float4((float)o.beta, 0.f, 0.f, 0.f);
      }
    } else if (KIND == J_T5) {
      T5Out o;
      if (live) pass = t5_candidate(s, g, ab.x, ab.y, &o, nullptr, nullptr, nullptr);
      if (pass) {
        st.p_d2[j] = make_double2(o.eta, o.phi);
        st.p_d2b[j] = make_double2(o.chi2, o.R);
        st.p_f4[j] = make_float4((float)o.pt, 0.f, 0.f, 0.f);
      }
    } else {
      double c2 = 0.0;
      if (live) pass = px_candidate<KIND>(geo, s, g, ab.x, ab.y, &c2);
      if (pass) st.p_d2[j] = make_double2(c2, 0.0);
    }
    if (pass) atomicOr(&st.mask[(size_t)(key / kItemCand) * kItemWords + ((key % kItemCand) >> 5)], 1u << (key & 31u));
  }
}
template <int KIND>
__global__ void __launch_bounds__(128, KIND == J_T3 ? 8 : 5) k_join_decide(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B,
                                                      const __grid_constant__ Params g) {
  pdl_enter();
  LST_SLOT(B);
  join_decide_body<KIND>(geo, s, g);
}
__global__ void __launch_bounds__(128, 8) k_px_decide(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B,
                                                    const __grid_constant__ Params g) {
  pdl_enter();
  LST_SLOT(B);
  if (blockIdx.y == 0) join_decide_body<J_PT5>(geo, s, g);
  else join_decide_body<J_PT3>(geo, s, g);
}

// One thread per pool entry: canonical position; constituent indices re-read from the inputs.  Then
// the level's CSR by first constituent: the objects of index row x (a first MD, or a pixel seed)
// start at the rank of the first candidate of the first join row that belongs to x.
template <int KIND>
__device__ __forceinline__ void join_fill_body(const SlotDev &s) {
  const int stage = JoinTraits<KIND>::stage;
  const StageBuf &st = s.st[stage];
  const Header *hdr = s.hdr;
  const uint32_t n_out = hdr->n_obj[JoinTraits<KIND>::out_level], n_items = hdr->n_items[stage];
  const uint32_t n_rows = hdr->n_obj[JoinTraits<KIND>::rows_level];
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nt = gridDim.x * blockDim.x;
  {
    const uint32_t n_idx = (KIND == J_T3 || KIND == J_T5) ? hdr->n_obj[0] : hdr->n_seeds;
    const uint32_t *in_off = KIND == J_T3 ? s.ls_md_off : (KIND == J_T5 ? s.t3_md_off : s.px_off);
    uint32_t *out_off = KIND == J_T3 ? s.t3_md_off : (KIND == J_T5 ? s.t5_md_off : (KIND == J_PT5 ? s.pt5_pls_off : s.pt3_pls_off));
    for (uint32_t x = tid; x <= n_idx; x += nt) {
      const uint32_t a = in_off[x];
      uint32_t off = n_out;
      if (a < n_rows && n_items) off = rank_before(st, n_items, n_out, st.g_item0[a / kRowChunk] * (uint32_t)kItemCand + st.row_cum[a]);
      out_off[x] = off;
    }
  }
  const uint32_t n = n_out ? min(hdr->cl_used[stage], st.cap_cl) : 0u;
  for (uint32_t j = tid; j < n; j += nt) {
    const uint32_t idx = pool_target(st, st.cl_key[j]);
    if (idx == 0xFFFFFFFFu) continue;
    const uint2 ab = st.cl_ab[j];
    if (KIND == J_T3) {
      const uint2 la = s.ls_md[ab.x], lb = s.ls_md[ab.y];
      s.t3_md[idx] = make_uint4(la.x, la.y, lb.y, 0u);
      s.t3_ls[idx] = ab;
      s.t3_kd[idx] = st.p_d2[j];
      st_f(s, s.t3_beta, idx, st.p_f4[j].x);
    } else if (KIND == J_T5) {
      const uint4 ta = s.t3_md[ab.x], tb = s.t3_md[ab.y];
      const uint32_t m[5] = {ta.x, ta.y, ta.z, tb.y, tb.z};
#pragma unroll
      for (int q = 0; q < 5; ++q) s.t5_md[(size_t)5 * idx + q] = m[q];
      const double2 cr = st.p_d2b[j];
      s.t5_t3[idx] = ab;
      s.t5_chi2[idx] = cr.x;
      s.t5_etaphi[idx] = st.p_d2[j];
      st_f4(s, s.t5_f, idx, make_float4((float)cr.y, (float)cr.x, (float)s.t3_kd[ab.x].x, (float)s.t3_kd[ab.y].x));
      st_f(s, s.t5_pt, idx, st.p_f4[j].x);
    } else {
      // S0, same-seed rule (k_dedup.cu): the seed's minimum score, on the bit pattern of the non-negative double
      const double c2 = st.p_d2[j].x;
      if (KIND == J_PT5) { s.pt5_po[idx] = ab; s.pt5_chi2[idx] = c2; }
      else { s.pt3_po[idx] = ab; s.pt3_chi2[idx] = c2; }
      atomicMin((KIND == J_PT5 ? s.pls_min5 : s.pls_min3) + ab.x, (unsigned long long)__double_as_longlong(c2));
    }
  }
}
template <int KIND>
__global__ void __launch_bounds__(256) k_join_fill(const __grid_constant__ Batch B) {
  pdl_enter();
  LST_SLOT(B);
  join_fill_body<KIND>(s);
}
__global__ void __launch_bounds__(256) k_px_fill(const __grid_constant__ Batch B) {
  pdl_enter();
  LST_SLOT(B);
  if (blockIdx.y == 0) join_fill_body<J_PT5>(s);
  else join_fill_body<J_PT3>(s);
}

// ------------------------------------------------------------------ launchers
template <int KIND>
static void launch_join_t(const Ctx &c, const Batch &b, uint32_t row_cap, uint32_t out_cap, cudaStream_t st) {
  const int gg = (int)((row_cap / kRowChunk + 1 + kJoinGroupWarps - 1) / kJoinGroupWarps);
  launch_k(c, st, JoinTraits<KIND>::n_groups, k_join_groups<KIND>, dim3(gg < c.n_sm * 8 ? gg : c.n_sm * 8), 32 * kJoinGroupWarps, 0,
           false, b);
  launch_k(c, st, JoinTraits<KIND>::n_eval, k_join_eval<KIND>, dim3(c.n_sm * 16), kThreads, 0, false, b, c.par);
  launch_k(c, st, JoinTraits<KIND>::n_decide, k_join_decide<KIND>, dim3(c.n_sm * 4), 128, 0, false, c.geo, b, c.par);
  launch_counts(c, b, JoinTraits<KIND>::stage, JoinTraits<KIND>::out_level, out_cap, false, st);
  launch_k(c, st, JoinTraits<KIND>::n_fill, k_join_fill<KIND>, dim3(c.n_sm * 4), 256, 0, false, b);
}

void launch_t3(const Ctx &c, const Batch &b, cudaStream_t st) { launch_join_t<J_T3>(c, b, b.s[0].cap_ls, b.s[0].cap_t3, st); }
void launch_t5(const Ctx &c, const Batch &b, cudaStream_t st) { launch_join_t<J_T5>(c, b, b.s[0].cap_t3, b.s[0].cap_t5, st); }

// pT5 (blockIdx.y = 0) and pT3 (1): independent of one another, the same five launches serve both
void launch_pixel_joins(const Ctx &c, const Batch &b, cudaStream_t st) {
  const uint32_t row_cap = b.s[0].cap_seeds * (uint32_t)kPxCap;
  const int gg = (int)((row_cap / kRowChunk + 1 + kJoinGroupWarps - 1) / kJoinGroupWarps);
  launch_k(c, st, "k_px_groups", k_px_groups, dim3(gg < c.n_sm * 4 ? gg : c.n_sm * 4, 2), 32 * kJoinGroupWarps, 0, false, b);
  launch_k(c, st, "k_px_eval", k_px_eval, dim3(c.n_sm * 8, 2), kThreads, 0, false, b, c.par);
  launch_k(c, st, "k_px_decide", k_px_decide, dim3(c.n_sm * 2, 2), 128, 0, false, c.geo, b, c.par);
  launch_counts(c, b, S_PT5, 5, b.s[0].cap_pt5, true, st);
  launch_k(c, st, "k_px_fill", k_px_fill, dim3(c.n_sm * 2, 2), 256, 0, false, b);
}

}  // namespace lst
